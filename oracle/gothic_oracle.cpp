/*
 * gothic_oracle.cpp -- CPU oracle for the GOTHIC hot path (Miki & Umemura, arxiv 1610.07279).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, step-by-step restatement of what
 * the paper's method computes, written from PAPER.md (cited as P:<line>) and the readings listed in
 * DESIGN.md (R1..R12).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call it.  It shares no code, header, table or helper with the CUDA path under
 * paper_1610_07279_b200/csrc/, and neither includes the other.
 *
 * Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC   (see oracle/build.py)
 * -ffp-contract=off matters: every fp32 expression that decides an integer (a key bit, a MAC outcome,
 * a time-step level) is written with explicit fmaf()/single operations and must not be re-fused.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"):
 *   direct sum            : eq. 1 vs numpy brute force, two-body closed form, cube symmetry
 *   encodePeano3D/decode  : bijection, face-adjacency ("one-stroke"), prefix hierarchy,
 *                           decode(encode) = id, level-1 table from
 *   Morton                : naive per-bit interleave
 *   sort                  : permutation / non-decreasing / stable
 *   tree                  : independent recursive builder + partition invariants
 *   moments               : numpy brute force (P:62 definitions)
 *   walk                  : Delta=0 equals eq. 1; error shrinks as Delta tightens;
 *                           Plummer closed form at large N; momentum;
 *                           eq. 5 / eq. 2 / eq. 3 written literally in pure-Python per-particle walks (r_crit = 0);
 *                           group a_min = min over members (R4): pure-Python group walk with |a_old| spread over four
 *                           decades + "group acceptance => eq. 5 holds for every member"
 *   levels / active set   : closed-form NFW level fractions; nesting invariants
 * Parity UNPINNED (report only): absolute error-vs-Delta values and interactions per step (the paper
 * gives them only as figures).
 */
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>
#include <utility>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef uint64_t PHint; /* "unsigned long int" when the key is longer than 30 bits */

static const int NLEV = 21; /* R1: 21 bits per axis -> 63-bit key */

/* ---- Listing 1, reconstructed: DESIGN.md reading G5 ------------------------------------ */
static PHint encodePeano3D(int Nlev, PHint px, PHint py, PHint pz)
{
    PHint key = 0;
    for (int jj = Nlev - 1; jj >= 0; jj--) {
        /* get xi, yi, and zi */
        PHint xi = (px >> jj) & 1;
        PHint yi = (py >> jj) & 1;
        PHint zi = (pz >> jj) & 1;
        /* turn px, py, and pz */
        px ^= -(xi & ((!yi) | zi));
        py ^= -((xi & (yi | zi)) | (yi & (!zi)));
        pz ^= -((xi & (!yi) & (!zi)) | (yi & (!zi)));
        /* append 3 bits to the key */
        key |= ((xi << 2) | ((xi ^ yi) << 1) | ((xi ^ zi) ^ yi)) << (3 * jj);
        if (zi) { /* rotate uncyclic (x->z->y->x) */
            PHint pt = px; px = py; py = pz; pz = pt;
        } else if (!yi) { /* exchange x and z */
            PHint pt = px; px = pz; pz = pt;
        }
    }
    return key;
}

/* ---- Listing 2, reconstructed: P:466 prints 3*jj+1 for zi (typo, must be 3*jj);
 *      the "append 1 bit" lines are lost and re-derived by inverting P:417 ---------------- */
static void decodePeano3D(int Nlev, PHint key, PHint *rx, PHint *ry, PHint *rz)
{
    PHint px = 0, py = 0, pz = 0;
    for (int jj = 0; jj < Nlev; jj++) {
        PHint xi = (key >> (3 * jj + 2)) & 1;
        PHint yi = (key >> (3 * jj + 1)) & 1;
        PHint zi = (key >> (3 * jj)) & 1;
        if (yi ^ zi) { /* rotate cyclic (x->y->z->x) */
            PHint pt = px; px = pz; pz = py; py = pt;
        } else if (((!xi) & (!yi) & (!zi)) || (xi & yi & zi)) { /* exchange x and z */
            PHint pt = px; px = pz; pz = pt;
        }
        PHint mask = ((PHint)1 << jj) - 1;
        px ^= mask & (-(xi & (yi | zi)));
        py ^= mask & (-((xi & ((!yi) | (!zi))) | ((!xi) & yi & zi)));
        pz ^= mask & (-((xi & (!yi) & (!zi)) | (yi & zi)));
        px |= xi << jj;          /* append 1 bit to the position: inverse of P:417 */
        py |= (xi ^ yi) << jj;
        pz |= (yi ^ zi) << jj;
    }
    *rx = px; *ry = py; *rz = pz;
}

/* ---- Listing 3: Morton key up to 63 bits by multiply-and-mask dilation -------------------- */
static PHint dilate3D(PHint val)
{
    val = (val * 0x100000001ULL) & 0x7fff00000000ffffULL;
    val = (val * 0x000010001ULL) & 0x00ff0000ff0000ffULL;
    val = (val * 0x000000101ULL) & 0x700f00f00f00f00fULL;
    val = (val * 0x000000011ULL) & 0x30c30c30c30c30c3ULL;
    val = (val * 0x000000005ULL) & 0x1249249249249249ULL;
    return val;
}
static PHint genMorton3D(PHint ix, PHint iy, PHint iz)
{
    return (dilate3D(ix) << 2) | (dilate3D(iy) << 1) | dilate3D(iz);
}

struct Box { float xmin, ymin, zmin, side; };

/* O1 / reading R1: root cube anchored at the per-axis minima, side = smallest power of two strictly
 * greater than the largest per-axis extent (side = 1 if the extent is 0). */
static Box root_box(const float *pos_m, uint32_t n)
{
    float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (uint32_t i = 0; i < n; i++)
        for (int k = 0; k < 3; k++) {
            float v = pos_m[4 * (size_t)i + k];
            lo[k] = std::min(lo[k], v);
            hi[k] = std::max(hi[k], v);
        }
    float ext = 0.0f;
    for (int k = 0; k < 3; k++) ext = std::max(ext, hi[k] - lo[k]);
    float side = 1.0f;
    if (ext > 0.0f) {
        int e;
        (void)frexpf(ext, &e); /* ext = f * 2^e, f in [0.5, 1)  =>  2^e > ext */
        side = ldexpf(1.0f, e);
    }
    Box b = {lo[0], lo[1], lo[2], side};
    return b;
}

/* O2: 21-bit integer coordinate: fp32 subtract, exact power-of-two scaling, truncate, clamp. */
static inline uint32_t grid_coord(float x, float xmin, float scale)
{
    float t = (x - xmin) * scale;
    float f = floorf(t);
    if (!(f > 0.0f)) return 0u;
    if (f >= 2097151.0f) return 2097151u;
    return (uint32_t)f;
}

extern "C" {

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

uint64_t oracle_encode_peano3d(int nlev, uint64_t x, uint64_t y, uint64_t z) { return encodePeano3D(nlev, x, y, z); }
void oracle_decode_peano3d(int nlev, uint64_t key, uint64_t *xyz) { decodePeano3D(nlev, key, xyz, xyz + 1, xyz + 2); }
uint64_t oracle_morton3d(uint64_t x, uint64_t y, uint64_t z) { return genMorton3D(x, y, z); }

void oracle_root_box(const float *pos_m, uint32_t n, float *box4)
{
    Box b = root_box(pos_m, n);
    box4[0] = b.xmin; box4[1] = b.ymin; box4[2] = b.zmin; box4[3] = b.side;
}

/* O2. key_kind 0 = Peano-Hilbert (paper default), 1 = Morton. */
void oracle_keys(const float *pos_m, uint32_t n, const float *box4, int key_kind, uint64_t *key)
{
    const float scale = 2097152.0f / box4[3];
    for (uint32_t i = 0; i < n; i++) {
        uint32_t ix = grid_coord(pos_m[4 * (size_t)i + 0], box4[0], scale);
        uint32_t iy = grid_coord(pos_m[4 * (size_t)i + 1], box4[1], scale);
        uint32_t iz = grid_coord(pos_m[4 * (size_t)i + 2], box4[2], scale);
        key[i] = key_kind == 0 ? encodePeano3D(NLEV, ix, iy, iz) : genMorton3D(ix, iy, iz);
    }
}

/* O3: stable sort of (key, original index) by key. */
void oracle_sort(const uint64_t *key, uint32_t n, uint64_t *key_sorted, uint32_t *perm)
{
    std::vector<uint32_t> idx(n);
    std::iota(idx.begin(), idx.end(), 0u);
    std::stable_sort(idx.begin(), idx.end(), [&](uint32_t a, uint32_t b) { return key[a] < key[b]; });
    for (uint32_t s = 0; s < n; s++) { perm[s] = idx[s]; key_sorted[s] = key[idx[s]]; }
}

/* O4 (reading R2): canonical oct-tree over the sorted keys, breadth-first ids.
 * Returns the node count, or -1 if it exceeds node_cap.  level_ofs has 23 entries:
 * level_ofs[L] = id of the first node of level L, level_ofs[n_levels..22] = n_nodes. */
int64_t oracle_build_tree(const uint64_t *key_sorted, uint32_t n, int n_leaf, uint32_t node_cap,
                          uint32_t *head, uint32_t *num, uint32_t *child, uint8_t *level, uint8_t *nchild,
                          uint32_t *level_ofs)
{
    struct Nd { uint32_t head, num; };
    std::vector<Nd> cur, nxt;
    uint64_t n_nodes = 0;
    cur.push_back({0u, n});
    for (int L = 0; L <= NLEV + 1; L++) level_ofs[L] = 0;
    int L = 0;
    for (; !cur.empty(); L++) {
        level_ofs[L] = (uint32_t)n_nodes;
        const uint64_t base = n_nodes;               /* ids of this level: base .. base+cur.size() */
        const uint64_t next_base = base + cur.size(); /* ids of the next level start here */
        if (next_base > node_cap) return -1;
        nxt.clear();
        for (size_t k = 0; k < cur.size(); k++) {
            const uint64_t id = base + k;
            head[id] = cur[k].head;
            num[id] = cur[k].num;
            level[id] = (uint8_t)L;
            if (cur[k].num > (uint32_t)n_leaf && L < NLEV) {
                /* children = maximal sub-ranges with equal key >> 3*(21-L-1), in key order;
                 * empty octants are not stored ("trimTree", Table 2) */
                const int sh = 3 * (NLEV - L - 1);
                child[id] = (uint32_t)(next_base + nxt.size());
                uint32_t s = cur[k].head, e = cur[k].head + cur[k].num, nc = 0;
                while (s < e) {
                    uint32_t t = s + 1;
                    while (t < e && (key_sorted[t] >> sh) == (key_sorted[s] >> sh)) t++;
                    nxt.push_back({s, t - s});
                    nc++;
                    s = t;
                }
                nchild[id] = (uint8_t)nc;
            } else {
                child[id] = 0xFFFFFFFFu;
                nchild[id] = 0;
            }
        }
        n_nodes = next_base;
        cur.swap(nxt);
    }
    for (int k = L; k <= NLEV + 1; k++) level_ofs[k] = (uint32_t)n_nodes;
    return (int64_t)n_nodes;
}

/* O5 (Fig. 1; reading R9): m_J = sum m_j, r_J = centre of mass, b_J = max |r_j - r_J| measured
 * from the fp32-rounded r_J that is stored.  Accumulates in double.  Nodes with num = 1 copy the particle. */
void oracle_moments(const float *pos_sorted, uint32_t n_nodes, const uint32_t *head, const uint32_t *num,
                    float *com4, float *b)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t J = 0; J < (int64_t)n_nodes; J++) {
        const uint32_t h = head[J], c = num[J];
        if (c == 1) {
            std::memcpy(com4 + 4 * J, pos_sorted + 4 * (size_t)h, 4 * sizeof(float));
            b[J] = 0.0f;
            continue;
        }
        double sx = 0, sy = 0, sz = 0, sm = 0;
        for (uint32_t j = h; j < h + c; j++) {
            const float *p = pos_sorted + 4 * (size_t)j;
            sx += (double)p[3] * p[0]; sy += (double)p[3] * p[1]; sz += (double)p[3] * p[2]; sm += p[3];
        }
        const float cx = (float)(sx / sm), cy = (float)(sy / sm), cz = (float)(sz / sm);
        double b2 = 0.0;
        for (uint32_t j = h; j < h + c; j++) {
            const float *p = pos_sorted + 4 * (size_t)j;
            const double dx = (double)p[0] - cx, dy = (double)p[1] - cy, dz = (double)p[2] - cz;
            b2 = std::max(b2, dx * dx + dy * dy + dz * dz);
        }
        com4[4 * J + 0] = cx; com4[4 * J + 1] = cy; com4[4 * J + 2] = cz; com4[4 * J + 3] = (float)sm;
        b[J] = (float)std::sqrt(b2);
    }
}

/* O5b (NEXT row f3; eq. 4): B_2 = sum_j m_j |r_j - r_J|^2 over the cell's particles about a GIVEN stored centre,
 * accumulated in double, rounded once. */
void oracle_b2(const float *pos_sorted, uint32_t n_nodes, const uint32_t *head, const uint32_t *num, const float *com4, float *B2)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t J = 0; J < (int64_t)n_nodes; J++) {
        double acc = 0.0;
        for (uint32_t j = head[J]; j < head[J] + num[J]; j++) {
            const float *p = pos_sorted + 4 * (size_t)j;
            const double dx = (double)p[0] - com4[4 * J], dy = (double)p[1] - com4[4 * J + 1], dz = (double)p[2] - com4[4 * J + 2];
            acc += (double)p[3] * (dx * dx + dy * dy + dz * dz);
        }
        B2[J] = (float)acc;
    }
}

/* O5, second half only: b_J = max |r_j - r_J| about a GIVEN stored centre com4 (stage-wise parity: the radius a
 * CUDA build reports is checked against the definition applied to the centre that same build stored). */
void oracle_radius(const float *pos_sorted, uint32_t n_nodes, const uint32_t *head, const uint32_t *num,
                   const float *com4, float *b)
{
#pragma omp parallel for schedule(dynamic, 256)
    for (int64_t J = 0; J < (int64_t)n_nodes; J++) {
        double b2 = 0.0;
        for (uint32_t j = head[J]; j < head[J] + num[J]; j++) {
            const float *p = pos_sorted + 4 * (size_t)j;
            const double dx = (double)p[0] - com4[4 * J], dy = (double)p[1] - com4[4 * J + 1], dz = (double)p[2] - com4[4 * J + 2];
            b2 = std::max(b2, dx * dx + dy * dy + dz * dz);
        }
        b[J] = (float)std::sqrt(b2);
    }
}

/* O6 (reading R6; criterion from BASELINE.json configs[2]): dt_i = eta sqrt(eps/|a_i|) floored to a power
 * of two.  q = dt^4 = c / |a|^2 with c = (float)(eta^4 eps^2) formed by the caller; exponent of dt =
 * floor(ilogb(q) / 4).  Levels count up from the finest present, clamped to max_levels - 1. */
static inline int dt_exponent(const float *a, float c)
{
    const float a2 = fmaf(a[2], a[2], fmaf(a[1], a[1], a[0] * a[0]));
    if (!(a2 > 0.0f)) return 127;          /* |a| = 0 (or NaN): coarsest */
    const float q = c / a2;
    if (std::isinf(q) || std::isnan(q)) return 127;
    if (q == 0.0f) return -38;             /* below the smallest subnormal: floor(-150/4) */
    const int e = ilogbf(q);               /* exact integer exponent, subnormals included */
    return (e >= 0) ? e / 4 : -((-e + 3) / 4); /* floor division */
}

void oracle_levels(const float *acc_pot, uint32_t n, float c, int max_levels, uint8_t *level, int32_t *emin_nlev)
{
    int emin = 1 << 30;
    std::vector<int> e(n);
    for (uint32_t i = 0; i < n; i++) { e[i] = dt_exponent(acc_pot + 4 * (size_t)i, c); emin = std::min(emin, e[i]); }
    int lmax = 0;
    for (uint32_t i = 0; i < n; i++) {
        int l = std::min(e[i] - emin, max_levels - 1);
        level[i] = (uint8_t)l;
        lmax = std::max(lmax, l);
    }
    emin_nlev[0] = n ? emin : 0;
    emin_nlev[1] = n ? lmax + 1 : 0;
}

/* O6: particle active at substep s (1-based) iff s mod 2^level == 0  <=>  level <= ctz(s). */
uint32_t oracle_active(const uint8_t *level, uint32_t n, uint32_t substep, uint32_t *active)
{
    uint32_t k = 0;
    for (uint32_t i = 0; i < n; i++) {
        const uint32_t period = 1u << level[i];
        if (substep % period == 0) active[k++] = i;
    }
    return k;
}

/* Eq. 1 in double, G = 1, with the potential of reading R5:
 * a_i = sum_{j != i} m_j (r_j - r_i) / (|r_j - r_i|^2 + eps^2)^{3/2},  Phi_i = - sum_{j != i} m_j / sqrt(...).
 * targets == NULL -> all particles.  out4: (ax, ay, az, Phi) per target. */
void oracle_direct(const float *pos_m, uint32_t n, const uint32_t *targets, uint32_t nt, double eps, double *out4)
{
    const double eps2 = eps * eps;
    const uint32_t m = targets ? nt : n;
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < (int64_t)m; t++) {
        const uint32_t i = targets ? targets[t] : (uint32_t)t;
        const double xi = pos_m[4 * (size_t)i], yi = pos_m[4 * (size_t)i + 1], zi = pos_m[4 * (size_t)i + 2];
        double ax = 0, ay = 0, az = 0, ph = 0;
        for (uint32_t j = 0; j < n; j++) {
            if (j == i) continue;
            const double dx = pos_m[4 * (size_t)j] - xi, dy = pos_m[4 * (size_t)j + 1] - yi, dz = pos_m[4 * (size_t)j + 2] - zi;
            const double r2 = dx * dx + dy * dy + dz * dz + eps2;
            const double u = 1.0 / std::sqrt(r2);
            const double mu3 = pos_m[4 * (size_t)j + 3] * u * u * u;
            ax += mu3 * dx; ay += mu3 * dy; az += mu3 * dz;
            ph -= pos_m[4 * (size_t)j + 3] * u;
        }
        out4[4 * t] = ax; out4[4 * t + 1] = ay; out4[4 * t + 2] = az; out4[4 * t + 3] = ph;
    }
}

void oracle_group_ball(const float *pos_sorted, const uint32_t *members, uint32_t k, int ball_kind, float *ball4);

static inline float dist2f(const float *a, const float *b)
{
    const float dx = a[0] - b[0], dy = a[1] - b[1], dz = a[2] - b[2];
    return fmaf(dz, dz, fmaf(dy, dy, dx * dx));
}

/* Centre of the pseudo i-particle's enclosing ball (App. B).  The radius is then always the exact maximum distance
 * of the members from that centre.
 *   ball_kind 0, GEO (item 3): centre of the bounding rectangular cuboid.
 *   ball_kind 1, EBS (item 2): Ritter's efficient bounding sphere (1990).  Pass 1: the first members (ascending order) that
 *     attain the minimum and the maximum of each coordinate; of the three pairs the one farthest apart (x before y before z on
 *     ties) spans the first sphere: centre = midpoint, radius = distance from the centre to the pair's maximum point.  Pass 2,
 *     members in ascending order: a point at distance dist > r grows the sphere just enough to contain it and the old sphere:
 *     r' = (r + dist)/2, centre moves by (dist - r')/dist of the way to the point.  fp32, operations as written (R17). */
static float ball_radius2(const float *pos_sorted, const uint32_t *members, uint32_t k, const float rI[3])
{
    float b2max = 0.0f;
    for (uint32_t q = 0; q < k; q++) b2max = std::max(b2max, dist2f(pos_sorted + 4 * (size_t)members[q], rI));
    return b2max;
}

/*   ball_kind 4, SEB (item 1): the smallest enclosing ball.  The paper names Fischer et al. (2003) and gives nothing else; the ball
 *     itself is unique, so any exact method serves.  Reading R19: Welzl's move-to-front recursion over the members in ascending
 *     order, single precision, operations as written.  A support set of m <= 4 points fixes the ball through them (m = 1 the point,
 *     2 the midpoint, 3 the circumcircle's centre in their plane, 4 the circumsphere: Cramer's rule about the first support point);
 *     a (near-)degenerate set (determinant <= 1e-12 of its scale) keeps the ball of the set without its last point.  A member counts
 *     as outside when its squared distance exceeds r^2 (1 + 2^-20).  As for the other balls the radius used by the walk is then the
 *     exact maximum distance of the members from the centre found, so rounding can cost tightness, never enclosure. */
struct SebBall { float c[3]; float r2; };

static SebBall seb_from_support(const float S[4][3], int m)
{
    SebBall B;
    B.c[0] = B.c[1] = B.c[2] = 0.0f;
    B.r2 = -1.0f;
    if (m == 0) return B;
    if (m == 1) { B.c[0] = S[0][0]; B.c[1] = S[0][1]; B.c[2] = S[0][2]; B.r2 = 0.0f; return B; }
    if (m == 2) {
        for (int d = 0; d < 3; d++) B.c[d] = 0.5f * (S[0][d] + S[1][d]);
        B.r2 = dist2f(S[0], B.c);
        return B;
    }
    const float a[3] = {S[1][0] - S[0][0], S[1][1] - S[0][1], S[1][2] - S[0][2]};
    const float b[3] = {S[2][0] - S[0][0], S[2][1] - S[0][1], S[2][2] - S[0][2]};
    const float aa = fmaf(a[2], a[2], fmaf(a[1], a[1], a[0] * a[0]));
    const float bb = fmaf(b[2], b[2], fmaf(b[1], b[1], b[0] * b[0]));
    const float ab = fmaf(a[2], b[2], fmaf(a[1], b[1], a[0] * b[0]));
    if (m == 3) {
        const float det = fmaf(aa, bb, -(ab * ab));
        if (!(det > 1e-12f * (aa * bb))) return seb_from_support(S, 2);
        const float l1 = (0.5f * (bb * (aa - ab))) / det, l2 = (0.5f * (aa * (bb - ab))) / det;
        float x[3];
        for (int d = 0; d < 3; d++) x[d] = fmaf(l2, b[d], l1 * a[d]);
        for (int d = 0; d < 3; d++) B.c[d] = S[0][d] + x[d];
        B.r2 = fmaf(x[2], x[2], fmaf(x[1], x[1], x[0] * x[0]));
        return B;
    }
    const float c[3] = {S[3][0] - S[0][0], S[3][1] - S[0][1], S[3][2] - S[0][2]};
    const float cc = fmaf(c[2], c[2], fmaf(c[1], c[1], c[0] * c[0]));
    /* b x c, c x a, a x b */
    const float bc[3] = {fmaf(b[1], c[2], -(b[2] * c[1])), fmaf(b[2], c[0], -(b[0] * c[2])), fmaf(b[0], c[1], -(b[1] * c[0]))};
    const float ca[3] = {fmaf(c[1], a[2], -(c[2] * a[1])), fmaf(c[2], a[0], -(c[0] * a[2])), fmaf(c[0], a[1], -(c[1] * a[0]))};
    const float axb[3] = {fmaf(a[1], b[2], -(a[2] * b[1])), fmaf(a[2], b[0], -(a[0] * b[2])), fmaf(a[0], b[1], -(a[1] * b[0]))};
    const float det = fmaf(a[2], bc[2], fmaf(a[1], bc[1], a[0] * bc[0]));
    if (!(fabsf(det) > 1e-12f * sqrtf(aa * bb * cc))) return seb_from_support(S, 3);
    const float h = 0.5f / det;
    float x[3];
    for (int d = 0; d < 3; d++) x[d] = h * fmaf(cc, axb[d], fmaf(bb, ca[d], aa * bc[d]));
    for (int d = 0; d < 3; d++) B.c[d] = S[0][d] + x[d];
    B.r2 = fmaf(x[2], x[2], fmaf(x[1], x[1], x[0] * x[0]));
    return B;
}

/* Welzl: smallest ball of pts[idx[0 .. n)] with the m points of S on its boundary; idx is reordered (move to front). */
static SebBall seb_mtf(const float (*pts)[3], uint8_t *idx, int n, float S[4][3], int m, int *budget)
{
    SebBall B = seb_from_support(S, m);
    if (m == 4) return B;
    for (int i = 0; i < n; i++) {
        const float *p = pts[idx[i]];
        if (B.r2 < 0.0f || dist2f(p, B.c) > B.r2 * (1.0f + 9.5367431640625e-07f)) {
            if (--(*budget) < 0) return B;                       /* cannot happen for points in general position */
            S[m][0] = p[0]; S[m][1] = p[1]; S[m][2] = p[2];
            B = seb_mtf(pts, idx, i, S, m + 1, budget);
            const uint8_t t = idx[i];
            for (int j = i; j > 0; j--) idx[j] = idx[j - 1];
            idx[0] = t;
        }
    }
    return B;
}

static void seb_centre(const float *pos_sorted, const uint32_t *members, uint32_t k, float rI[3])
{
    float pts[64][3];
    uint8_t idx[64];
    const int n = (int)std::min<uint32_t>(k, 64u);
    for (int q = 0; q < n; q++) {
        for (int d = 0; d < 3; d++) pts[q][d] = pos_sorted[4 * (size_t)members[q] + d];
        idx[q] = (uint8_t)q;
    }
    float S[4][3];
    int budget = 4096;
    const SebBall B = seb_mtf(pts, idx, n, S, 0, &budget);
    rI[0] = B.c[0]; rI[1] = B.c[1]; rI[2] = B.c[2];
}

/*   ball_kind 2, COM (item 4): centre of mass of the members, sums over the members in ascending order with one fmaf each, then
 *     one division per coordinate.
 *   ball_kind 3, CMP (item 5): the smaller of the GEO and COM balls (GEO on ties). */
static void ball_centre(const float *pos_sorted, const uint32_t *members, uint32_t k, int ball_kind, float rI[3])
{
    if (ball_kind == 4) { seb_centre(pos_sorted, members, k, rI); return; }
    if (ball_kind == 2 || ball_kind == 3) {
        float sx = 0.0f, sy = 0.0f, sz = 0.0f, sm = 0.0f;
        for (uint32_t q = 0; q < k; q++) {
            const float *p = pos_sorted + 4 * (size_t)members[q];
            sx = fmaf(p[3], p[0], sx); sy = fmaf(p[3], p[1], sy); sz = fmaf(p[3], p[2], sz); sm += p[3];
        }
        float com[3] = {sx / sm, sy / sm, sz / sm};
        if (!(sm > 0.0f)) ball_centre(pos_sorted, members, k, 0, com);          /* massless members: fall back to GEO */
        if (ball_kind == 3) {
            float geo[3];
            ball_centre(pos_sorted, members, k, 0, geo);
            if (ball_radius2(pos_sorted, members, k, geo) <= ball_radius2(pos_sorted, members, k, com)) { com[0] = geo[0]; com[1] = geo[1]; com[2] = geo[2]; }
        }
        rI[0] = com[0]; rI[1] = com[1]; rI[2] = com[2];
        return;
    }
    if (ball_kind == 0) {
        float lo[3] = {INFINITY, INFINITY, INFINITY}, hi[3] = {-INFINITY, -INFINITY, -INFINITY};
        for (uint32_t q = 0; q < k; q++)
            for (int d = 0; d < 3; d++) {
                lo[d] = std::min(lo[d], pos_sorted[4 * (size_t)members[q] + d]);
                hi[d] = std::max(hi[d], pos_sorted[4 * (size_t)members[q] + d]);
            }
        for (int d = 0; d < 3; d++) rI[d] = 0.5f * (lo[d] + hi[d]);
        return;
    }
    uint32_t imin[3] = {0, 0, 0}, imax[3] = {0, 0, 0};
    for (uint32_t q = 1; q < k; q++)
        for (int d = 0; d < 3; d++) {
            const float v = pos_sorted[4 * (size_t)members[q] + d];
            if (v < pos_sorted[4 * (size_t)members[imin[d]] + d]) imin[d] = q;
            if (v > pos_sorted[4 * (size_t)members[imax[d]] + d]) imax[d] = q;
        }
    int a = 0;
    float best = -1.0f;
    for (int d = 0; d < 3; d++) {
        const float s2 = dist2f(pos_sorted + 4 * (size_t)members[imax[d]], pos_sorted + 4 * (size_t)members[imin[d]]);
        if (s2 > best) { best = s2; a = d; }
    }
    const float *pa = pos_sorted + 4 * (size_t)members[imin[a]], *pb = pos_sorted + 4 * (size_t)members[imax[a]];
    for (int d = 0; d < 3; d++) rI[d] = 0.5f * (pa[d] + pb[d]);
    float r2 = dist2f(pb, rI), r = sqrtf(r2);
    for (uint32_t q = 0; q < k; q++) {
        const float *p = pos_sorted + 4 * (size_t)members[q];
        const float dx = p[0] - rI[0], dy = p[1] - rI[1], dz = p[2] - rI[2];
        const float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        if (d2 > r2) {
            const float dist = sqrtf(d2), rn = 0.5f * (r + dist), f = (dist - rn) / dist;
            rI[0] = fmaf(f, dx, rI[0]); rI[1] = fmaf(f, dy, rI[1]); rI[2] = fmaf(f, dz, rI[2]);
            r = rn; r2 = rn * rn;
        }
    }
}

/* O7 (P:105-118 traversal with a pseudo i-particle; eq. 5; eq. 2; P:62 monopole).
 * One group = aligned chunk of G consecutive sorted indices (reading R3); members = its active particles;
 * GEO enclosing ball and a_min = min |a_old| over members (R4).  All MAC-deciding arithmetic in fp32 with
 * the operation order written here; the sums over the interaction list are in double.
 *   active == NULL  -> all n particles active.
 *   out4: double (ax, ay, az, Phi) for every sorted index (only active entries written).
 *   counts[0] += sum over groups |K| * |list|   (interactions, P:331 convention)
 *   counts[1] += MAC evaluations, counts[2] += groups walked, counts[3] += sum |list|
 *   group_lo/group_hi: only groups g with group_lo <= g < group_hi are walked (bounded samples).
 *   r_crit: "critical separation ... to judge whether to unify i-particles into a group or not" (§2.4).
 *           The paper gives no formula; reading R13: a chunk's member list (ascending sorted index) whose GEO ball has
 *           b_I > r_crit is cut into its first ceil(k/2) members and the rest, recursively, until b_I <= r_crit or one
 *           member is left; every piece then walks the tree on its own.  r_crit = INFINITY: no splitting (R3 as is). */
void oracle_walk(const float *pos_sorted, uint32_t n,
                 const uint32_t *head, const uint32_t *num, const uint32_t *child, const uint8_t *nchild,
                 const float *com4, const float *bJ, const float *B2 /* eq. 4; needed iff mac_kind == 2 */,
                 const uint32_t *active, uint32_t n_active, int G,
                 float eps, int mac_kind, float mac_param, const float *aold,
                 uint32_t group_lo, uint32_t group_hi, float r_crit, int ball_kind /* 0 GEO, 1 EBS, 2 COM, 3 CMP (App. B) */,
                 double *out4, uint64_t *counts)
{
    const uint32_t n_groups = (n + (uint32_t)G - 1) / (uint32_t)G;
    group_hi = std::min(group_hi, n_groups);
    /* members per group from the ascending active list */
    std::vector<uint32_t> first(n_groups + 1, 0);
    if (active) {
        for (uint32_t k = 0; k < n_active; k++) first[active[k] / G + 1]++;
        for (uint32_t g = 0; g < n_groups; g++) first[g + 1] += first[g];
    }
    const double eps2 = (double)eps * (double)eps;
    uint64_t c_int = 0, c_mac = 0, c_grp = 0, c_list = 0;

#pragma omp parallel for schedule(dynamic, 16) reduction(+ : c_int, c_mac, c_grp, c_list)
    for (int64_t g = group_lo; g < (int64_t)group_hi; g++) {
        std::vector<uint32_t> K;
        if (active) {
            for (uint32_t k = first[g]; k < first[g + 1]; k++) K.push_back(active[k]);
        } else {
            for (uint32_t s = (uint32_t)g * G; s < std::min(n, (uint32_t)(g + 1) * G); s++) K.push_back(s);
        }
        if (K.empty()) continue;
        /* §2.4 / R13: pieces of the member list, produced depth-first (first half before second half) */
        std::vector<std::pair<uint32_t, uint32_t>> todo(1, std::make_pair(0u, (uint32_t)K.size())), pieces;
        while (!todo.empty()) {
            const std::pair<uint32_t, uint32_t> pr = todo.back();
            todo.pop_back();
            const uint32_t cnt = pr.second - pr.first;
            float ball[4];
            oracle_group_ball(pos_sorted, K.data() + pr.first, cnt, ball_kind, ball);
            if (cnt > 1 && ball[3] > r_crit) {
                const uint32_t mid = pr.first + (cnt + 1) / 2;
                todo.push_back(std::make_pair(mid, pr.second));
                todo.push_back(std::make_pair(pr.first, mid));
            } else pieces.push_back(pr);
        }
        const std::vector<uint32_t> Kall = K;
        for (const std::pair<uint32_t, uint32_t> &pc : pieces) {
        K.assign(Kall.begin() + pc.first, Kall.begin() + pc.second);
        /* pseudo i-particle: enclosing ball (App. B; GEO item 3 or EBS item 2) and a_min over the members */
        float amin = INFINITY;
        if (aold) for (uint32_t k : K) amin = std::min(amin, aold[k]);
        float rI[3];
        ball_centre(pos_sorted, K.data(), (uint32_t)K.size(), ball_kind, rI);
        float b2max = 0.0f;
        for (uint32_t k : K) {
            const float dx = pos_sorted[4 * (size_t)k] - rI[0], dy = pos_sorted[4 * (size_t)k + 1] - rI[1],
                        dz = pos_sorted[4 * (size_t)k + 2] - rI[2];
            b2max = std::max(b2max, fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
        }
        const float bI = sqrtf(b2max);
        const float thr = mac_kind == 0 ? mac_param * amin : mac_param; /* Delta_acc * a_min (G = 1), or theta */

        /* traversal: pending set handled as a stack ("any order", R10) */
        std::vector<uint32_t> pending(1, 0u);
        std::vector<uint32_t> cells, parts; /* accepted cells; particles of opened leaves */
        while (!pending.empty()) {
            const uint32_t J = pending.back();
            pending.pop_back();
            c_mac++;
            const float dx = com4[4 * (size_t)J] - rI[0], dy = com4[4 * (size_t)J + 1] - rI[1], dz = com4[4 * (size_t)J + 2] - rI[2];
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const float d = fmaxf(sqrtf(r2) - bI, 0.0f); /* eq. 6-7: lambda * r_JI */
            bool accept = false;
            if (d > 0.0f) {
                if (mac_kind == 0) {
                    const float mb2 = (com4[4 * (size_t)J + 3] * bJ[J]) * bJ[J];
                    accept = thr * ((d * d) * (d * d)) >= mb2; /* eq. 5, both sides to the 4th power */
                } else if (mac_kind == 1) {
                    accept = bJ[J] <= thr * d;                 /* eq. 2 */
                } else {
                    /* eq. 3: d >= b/2 + sqrt(b^2/4 + sqrt(3 B_2 / Delta_mul)).  Since the right side is >= b, squaring
                     * d - b/2 gives d (d - b) >= sqrt(3 B_2 / Delta), i.e. d >= b and Delta (d (d - b))^2 >= 3 B_2: the form
                     * both sides evaluate in fp32 (R16; equivalence pinned in tests/test_oracle_multipole.py). */
                    const float t = d * (d - bJ[J]);
                    accept = d >= bJ[J] && thr * (t * t) >= 3.0f * B2[J];
                }
            }
            if (accept) cells.push_back(J);
            else if (child[J] == 0xFFFFFFFFu) {
                for (uint32_t s = head[J]; s < head[J] + num[J]; s++) parts.push_back(s);
            } else {
                for (uint32_t c = 0; c < nchild[J]; c++) pending.push_back(child[J] + c);
            }
        }
        /* evaluate: every member against every list entry (eq. 1 with pseudo j-particles, monopole) */
        for (uint32_t i : K) {
            const double xi = pos_sorted[4 * (size_t)i], yi = pos_sorted[4 * (size_t)i + 1], zi = pos_sorted[4 * (size_t)i + 2];
            double ax = 0, ay = 0, az = 0, ph = 0;
            for (uint32_t J : cells) {
                const double dx = com4[4 * (size_t)J] - xi, dy = com4[4 * (size_t)J + 1] - yi, dz = com4[4 * (size_t)J + 2] - zi;
                const double u = 1.0 / std::sqrt(dx * dx + dy * dy + dz * dz + eps2);
                const double mu3 = com4[4 * (size_t)J + 3] * u * u * u;
                ax += mu3 * dx; ay += mu3 * dy; az += mu3 * dz; ph -= com4[4 * (size_t)J + 3] * u;
            }
            for (uint32_t s : parts) {
                if (s == i) continue; /* j != i (eq. 1); reading R5 */
                const double dx = pos_sorted[4 * (size_t)s] - xi, dy = pos_sorted[4 * (size_t)s + 1] - yi, dz = pos_sorted[4 * (size_t)s + 2] - zi;
                const double u = 1.0 / std::sqrt(dx * dx + dy * dy + dz * dz + eps2);
                const double mu3 = pos_sorted[4 * (size_t)s + 3] * u * u * u;
                ax += mu3 * dx; ay += mu3 * dy; az += mu3 * dz; ph -= pos_sorted[4 * (size_t)s + 3] * u;
            }
            out4[4 * (size_t)i] = ax; out4[4 * (size_t)i + 1] = ay; out4[4 * (size_t)i + 2] = az; out4[4 * (size_t)i + 3] = ph;
        }
        const uint64_t L = cells.size() + parts.size();
        c_int += (uint64_t)K.size() * L;
        c_list += L;
        c_grp++;
        } /* pieces */
    }
    if (counts) { counts[0] += c_int; counts[1] += c_mac; counts[2] += c_grp; counts[3] += c_list; }
}

/* P:118 pin helper: for one group, the ball (r_I, b_I) exactly as oracle_walk forms it. */
void oracle_group_ball(const float *pos_sorted, const uint32_t *members, uint32_t k, int ball_kind, float *ball4)
{
    float rI[3];
    ball_centre(pos_sorted, members, k, ball_kind, rI);
    float b2max = 0.0f;
    for (uint32_t q = 0; q < k; q++) {
        const float dx = pos_sorted[4 * (size_t)members[q]] - rI[0], dy = pos_sorted[4 * (size_t)members[q] + 1] - rI[1],
                    dz = pos_sorted[4 * (size_t)members[q] + 2] - rI[2];
        b2max = std::max(b2max, fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
    }
    ball4[0] = rI[0]; ball4[1] = rI[1]; ball4[2] = rI[2]; ball4[3] = sqrtf(b2max);
}

/* O8 (NEXT row f1; section 2.7, eq. 15-17): second-order predictor-corrector under block time steps.
 * Every particle j carries its state (r, v, a) at its own last corrected time t_last[j], counted in units of dt_unit
 * (the finest step 2^e_min, so the float product below is exact).  Prediction of ALL j-particles to t_now:
 *   dt = (t_now - t_last[j]) dt_unit;  v^{n+1/2} = v^n + (dt/2) a^n  (eq. 15);  r^{n+1} = r^n + dt v^{n+1/2}  (eq. 16).
 * Single precision, one fused multiply-add per component, in this order (R15). */
void oracle_predict(const float *pos_m, const float *vel, const float *acc_pot, const uint32_t *t_last, uint32_t t_now,
                    float dt_unit, uint32_t n, float *pos_pred)
{
    for (uint32_t j = 0; j < n; j++) {
        const float dt = (float)(t_now - t_last[j]) * dt_unit;
        const float h = 0.5f * dt;
        for (int k = 0; k < 3; k++) {
            const float vh = fmaf(h, acc_pot[4 * (size_t)j + k], vel[4 * (size_t)j + k]);        /* eq. 15 */
            pos_pred[4 * (size_t)j + k] = fmaf(dt, vh, pos_m[4 * (size_t)j + k]);                /* eq. 16 */
        }
        pos_pred[4 * (size_t)j + 3] = pos_m[4 * (size_t)j + 3];                                  /* mass */
    }
}

/* Correction of the active i-particles (eq. 17): v^{n+1} = v^{n+1/2} + (dt/2) a^{n+1}, with v^{n+1/2} of eq. 15 over the
 * particle's own full step; the predicted position becomes the particle's position, a^{n+1} its acceleration and t_now its
 * time.  Level migration (the paper is silent; reading R15): the level wanted by the new acceleration is
 * clamp(dt_exponent(a^{n+1}) - e_min, 0, max_levels - 1); a particle may move to any FINER level at once, and ONE level coarser
 * only when t_now is a multiple of that coarser step (so that every particle stays aligned with its block).  level == NULL: none. */
void oracle_correct(const uint32_t *active, uint32_t n_active, const float *pos_pred, const float *acc_new, uint32_t t_now,
                    float dt_unit, float *pos_m, float *vel, float *acc_pot, uint32_t *t_last, uint8_t *level, float c,
                    int e_min, int max_levels)
{
    for (uint32_t q = 0; q < n_active; q++) {
        const size_t i = active[q];
        const float dt = (float)(t_now - t_last[i]) * dt_unit;
        const float h = 0.5f * dt;
        for (int k = 0; k < 3; k++) {
            const float vh = fmaf(h, acc_pot[4 * i + k], vel[4 * i + k]);                         /* eq. 15 */
            vel[4 * i + k] = fmaf(h, acc_new[4 * i + k], vh);                                    /* eq. 17 */
        }
        for (int k = 0; k < 4; k++) { pos_m[4 * i + k] = pos_pred[4 * i + k]; acc_pot[4 * i + k] = acc_new[4 * i + k]; }
        t_last[i] = t_now;
        if (level) {
            int want = dt_exponent(acc_new + 4 * i, c) - e_min;
            want = std::max(0, std::min(want, max_levels - 1));
            const int cur = level[i];
            if (want < cur) level[i] = (uint8_t)want;
            else if (want > cur && t_now % (1u << (cur + 1)) == 0) level[i] = (uint8_t)(cur + 1);
        }
    }
}

} /* extern "C" */
