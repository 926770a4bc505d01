"""-m gpu: the studies module runs end to end on small inputs and reports what the paper leads one to
expect: Hilbert order gives tighter groups and fewer interactions than Morton; interactions grow with the steps since
the tree was built when only the moments are refreshed."""
import json

import pytest

pytestmark = pytest.mark.gpu


def _lines(capsys):
    return [json.loads(l) for l in capsys.readouterr().out.splitlines() if l.startswith("{")]


def test_keys_study(capsys):
    from paper_1610_07279_b200 import studies
    studies.study_keys(1 << 16)
    r = {d["key"]: d for d in _lines(capsys)}
    assert r["peano_hilbert"]["group_ball_radius_median"] < r["morton"]["group_ball_radius_median"]
    assert r["peano_hilbert"]["interactions_unsplit"] < r["morton"]["interactions_unsplit"]      # whole 32-chunks: the order alone
    assert r["peano_hilbert"]["n_nodes"] == r["morton"]["n_nodes"]          # the same oct-tree, another order


def test_refresh_study(capsys):
    from paper_1610_07279_b200 import studies
    studies.study_refresh(1 << 15, 8)
    rows = _lines(capsys)
    rebuilt = {d["step"]: d["interactions"] for d in rows if d["mode"] == "rebuild_every_step"}
    kept = {d["step"]: d["interactions"] for d in rows if d["mode"] == "moments_only"}
    assert kept[8] > kept[4] > kept[1] and kept[8] > 1.05 * rebuilt[8]
    assert abs(rebuilt[8] - rebuilt[1]) < 0.05 * rebuilt[1]


def test_balls_study(capsys):
    from paper_1610_07279_b200 import studies
    studies.study_balls(1 << 15)
    rows = _lines(capsys)
    assert len(rows) == 60          # 5 balls x 3 MACs x 4 parameters
    for mac in ("acceleration", "multipole", "opening_angle"):
        geo = [d for d in rows if d["ball"] == "GEO" and d["mac"] == mac]
        assert all(b["err_median"] < a["err_median"] and b["interactions"] > a["interactions"] for a, b in zip(geo, geo[1:]))
    # the smallest ball opens the fewest cells (App. B: "the best choice is the SEB, which has the minimum radius")
    for a, b in zip([d for d in rows if d["ball"] == "SEB" and d["mac"] == "acceleration"], [d for d in rows if d["ball"] == "GEO" and d["mac"] == "acceleration"]):
        assert a["param"] == b["param"] and a["interactions"] <= b["interactions"]
