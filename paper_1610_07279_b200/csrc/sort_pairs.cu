// B3: stable LSD radix sort of (63-bit key, 32-bit index) pairs (the paper calls
// cub::DeviceRadixSort::SortPairs).  Hand-written one-sweep sort for sm_100a:
//
//   k_sort_hist      one pass over the keys -> the 8 digit histograms (8 bits per digit, 63 significant bits),
//   k_sort_scan      exclusive scan of each histogram = where every digit's run starts in the output of its pass,
//   k_sort_onesweep  one launch per digit, least significant first.  A CTA takes the next tile of 3072 pairs (ticket
//                    from an atomic counter, so that every earlier tile is already running), ranks its keys by
//                    digit (warp-private counters + match.any, items in index order => stable), publishes its digit
//                    counts, finds the sum over all earlier tiles by decoupled look-back (each of the 256 threads
//                    chases one digit: aggregate -> inclusive flags in one 32-bit word with the count), regroups
//                    keys and values by digit in shared memory and writes every run out contiguously.
//
// Per pass every pair is read once and written once (12 B each way): the HBM floor of an LSD radix sort.  Ties keep
// ascending original index (LSD passes are stable), which is what makes perm bit-exact against the oracle's
// std::stable_sort.
//
// Five passes instead of eight.  The low 23 bits of a key (the last 7 2/3 octal digits: cells of 2^-13.3 of the root cube) order
// particles only inside runs of equal upper 40 bits, and such runs are short (most particles are alone in theirs).  So the LSD
// passes cover bits 23..62 only, and
//   k_sort_fix_short  finds the runs and finishes the ones of up to 32 keys by a stable insertion sort on the low bits (one thread
//                     per run; nothing to do when the run is already in order, e.g. coincident particles),
//   k_sort_fix_long   finishes runs of 33 .. FIX_LONG_MAX keys by a stable rank sort in shared memory (one CTA per run).
// A longer run that is out of order raises flags[3]; gothic_build_tree then repeats the build with all eight passes (a pathological
// input: thousands of distinct particles inside one cell of 2^-13 of the box).
#include "gothic_ctx.cuh"

namespace {

constexpr int RADIX = 256;
constexpr int NPASS = 8;                    // 8 x 8 bits >= 63 (the full sort; the fast path runs the upper NPASS_FAST digits)
constexpr int NPASS_FAST = 5;
constexpr int LOW_BITS = 63 - 8 * NPASS_FAST;          // 23 bits left to the fix-up kernels
constexpr int FIX_SHORT_MAX = 32;
constexpr int FIX_LONG_MAX = 2048;
constexpr int SORT_TPB = 256;
constexpr int SORT_WARPS = SORT_TPB / 32;
#ifndef GOTHIC_SORT_IPT
#define GOTHIC_SORT_IPT 12
#endif
#ifndef GOTHIC_SORT_CTAS
#define GOTHIC_SORT_CTAS 4
#endif
constexpr int IPT = GOTHIC_SORT_IPT;        // items per thread
constexpr int TILE = SORT_TPB * IPT;        // pairs per CTA (3072: four CTAs of 256 threads per SM)
constexpr uint32_t ST_AGG = 1u << 30;       // status word: this tile's own count is in the low 30 bits
constexpr uint32_t ST_INC = 1u << 31;       //              the count of this and ALL earlier tiles is
constexpr uint32_t ST_VAL = ST_AGG - 1u;
constexpr uint32_t FULL = 0xffffffffu;

// scratch layout (u32 words): ghist[NPASS][RADIX] | ticket[NPASS] (+ pad to 16) | status[NPASS][ntiles][RADIX]
__host__ __device__ inline size_t sort_words_head() { return (size_t)NPASS * RADIX + 16; }

__global__ void __launch_bounds__(SORT_TPB) k_sort_hist(const uint64_t *__restrict__ key, uint32_t n, uint32_t *__restrict__ ghist, int shift0, int npass)
{
    __shared__ uint32_t s_h[NPASS][RADIX];
    for (int i = threadIdx.x; i < NPASS * RADIX; i += SORT_TPB) (&s_h[0][0])[i] = 0u;
    __syncthreads();
    const uint32_t stride = gridDim.x * SORT_TPB;
    for (uint32_t i = blockIdx.x * SORT_TPB + threadIdx.x; i < n; i += stride) {
        const uint64_t k = __ldg(key + i) >> shift0;
#pragma unroll
        for (int p = 0; p < NPASS; p++)
            if (p < npass) atomicAdd(&s_h[p][(uint32_t)(k >> (8 * p)) & 255u], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NPASS * RADIX; i += SORT_TPB) {
        const uint32_t v = (&s_h[0][0])[i];
        if (v) atomicAdd(ghist + i, v);
    }
}

// one CTA per pass: ghist[p][d] <- number of keys whose digit p is smaller than d
__global__ void __launch_bounds__(RADIX) k_sort_scan(uint32_t *__restrict__ ghist)
{
    __shared__ uint32_t s_w[RADIX / 32];
    uint32_t *h = ghist + blockIdx.x * RADIX;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t v = h[threadIdx.x];
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(FULL, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    uint32_t base = 0;
    for (uint32_t w = 0; w < warp; w++) base += s_w[w];
    h[threadIdx.x] = base + incl - v;
}

struct SortSmem {
    uint64_t keys[TILE];                    // the tile regrouped by digit
    uint32_t vals[TILE];
    uint32_t hist[SORT_WARPS][RADIX];       // per-warp digit counters, then exclusive offsets across the warps
    uint32_t dstart[RADIX];                 // where each digit's run starts inside the regrouped tile
    uint32_t gbase[RADIX];                  // global position of slot j of digit d = gbase[d] + j
    uint32_t wsum[SORT_WARPS];
    uint32_t tile;
};

__global__ void __launch_bounds__(SORT_TPB, GOTHIC_SORT_CTAS) k_sort_onesweep(const uint64_t *__restrict__ kin, const uint32_t *__restrict__ vin,
                                                            uint64_t *__restrict__ kout, uint32_t *__restrict__ vout, uint32_t n, int shift,
                                                            const uint32_t *__restrict__ gstart, uint32_t *__restrict__ ticket,
                                                            volatile uint32_t *status)
{
    extern __shared__ __align__(16) unsigned char s_raw[];
    SortSmem &S = *reinterpret_cast<SortSmem *>(s_raw);
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t lt = (1u << lane) - 1u;

    if (tid == 0) S.tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < SORT_WARPS * RADIX; i += SORT_TPB) (&S.hist[0][0])[i] = 0u;
    __syncthreads();
    const uint32_t tile = S.tile;
    const uint32_t base = tile * (uint32_t)TILE;
    const uint32_t n_valid = min((uint32_t)TILE, n - base);

    // ---- load: warp w owns the 512 consecutive pairs [512 w, 512 w + 512) of the tile, 32 at a time ----
    uint64_t k[IPT];
    uint32_t v[IPT];
#pragma unroll
    for (int i = 0; i < IPT; i++) {
        const uint32_t j = warp * (32u * IPT) + (uint32_t)i * 32u + lane;
        k[i] = j < n_valid ? __ldg(kin + base + j) : ~0ull;
        v[i] = j < n_valid ? (vin ? __ldg(vin + base + j) : base + j) : 0u;
    }
    // ---- rank inside (warp, digit), in index order ----
    uint32_t pos[IPT];
#pragma unroll
    for (int i = 0; i < IPT; i++) {
        const uint32_t j = warp * (32u * IPT) + (uint32_t)i * 32u + lane;
        const bool valid = j < n_valid;
        const uint32_t d = (uint32_t)(k[i] >> shift) & 255u;
        // the lanes of the row with the same digit: eight ballots (one per digit bit) instead of match.any, which is the slower of the two here
        uint32_t peers = __ballot_sync(FULL, valid);
        if (!valid) peers = ~peers;
#pragma unroll
        for (int b = 0; b < 8; b++) {
            const uint32_t vote = __ballot_sync(FULL, (d >> b) & 1u);
            peers &= ((d >> b) & 1u) ? vote : ~vote;
        }
        const int leader = __ffs(peers) - 1;
        // one returning shared-memory atomic per distinct digit of the row: atomics of one warp on one address complete in
        // program order, so the rows need no barrier between them and their latencies overlap
        uint32_t old = 0;
        if ((int)lane == leader && valid) old = atomicAdd(&S.hist[warp][d], (uint32_t)__popc(peers));
        old = __shfl_sync(FULL, old, leader);
        pos[i] = old + __popc(peers & lt);
    }
    __syncthreads();

    // ---- thread t = digit t: offsets across the warps, run starts inside the tile, look-back over earlier tiles ----
    {
        uint32_t count = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; w++) {
            const uint32_t c = S.hist[w][tid];
            S.hist[w][tid] = count;
            count += c;
        }
        volatile uint32_t *st = status + (size_t)tile * RADIX + tid;
        if (tile == 0) *st = count | ST_INC;
        else *st = count | ST_AGG;
        // exclusive scan of the counts over the digits
        uint32_t incl = count;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(FULL, incl, o);
            if (lane >= (uint32_t)o) incl += y;
        }
        if (lane == 31) S.wsum[warp] = incl;
        __syncthreads();
        uint32_t wbase = 0;
        for (uint32_t w = 0; w < warp; w++) wbase += S.wsum[w];
        const uint32_t excl = wbase + incl - count;
        S.dstart[tid] = excl;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; w++) S.hist[w][tid] += excl;       // slot of (warp, digit, rank) = hist[warp][digit] + rank
        // decoupled look-back: sum of this digit's counts over tiles tile-1, tile-2, ... until an inclusive one
        uint32_t prefix = 0;
        if (tile > 0) {
            // four earlier tiles per step: their status words are independent loads, so a step costs one L2 round trip, not four
            int t = (int)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t sw[4];
#pragma unroll
                for (int q = 0; q < 4; q++) sw[q] = t - q >= 0 ? status[(size_t)(t - q) * RADIX + tid] : 0x80000000u;
#pragma unroll
                for (int q = 0; q < 4; q++) {
                    if (done) break;
                    if (sw[q] & ST_INC) { prefix += sw[q] & ST_VAL; done = true; }
                    else if (sw[q] & ST_AGG) { prefix += sw[q] & ST_VAL; t--; }
                    else { __nanosleep(20); break; }        // not published yet: look again from this tile
                }
            }
            *st = (prefix + count) | ST_INC;
        }
        S.gbase[tid] = gstart[tid] + prefix - excl;
    }
    __syncthreads();

    // ---- regroup by digit in shared memory ----
#pragma unroll
    for (int i = 0; i < IPT; i++) {
        const uint32_t j = warp * (32u * IPT) + (uint32_t)i * 32u + lane;
        if (j < n_valid) {
            const uint32_t d = (uint32_t)(k[i] >> shift) & 255u;
            const uint32_t p = S.hist[warp][d] + pos[i];
            S.keys[p] = k[i];
            S.vals[p] = v[i];
        }
    }
    __syncthreads();
    // ---- write every run out contiguously ----
#pragma unroll
    for (int i = 0; i < IPT; i++) {
        const uint32_t j = tid + (uint32_t)i * SORT_TPB;
        if (j < n_valid) {
            const uint64_t key = S.keys[j];
            const uint32_t dst = S.gbase[(uint32_t)(key >> shift) & 255u] + j;
            kout[dst] = key;
            vout[dst] = S.vals[j];
        }
    }
}

// Is the run of equal upper bits that holds entry i longer than FIX_LONG_MAX?  Two probes half that far away answer "no" for almost every
// caller (a run of more than 2 H entries reaches at least H to one side of each of its members); only then are the run's ends found by
// bisection on the upper bits, which the fast passes have fully sorted.  Reads upper bits only: k_sort_fix_short never changes those.
__device__ __forceinline__ bool run_too_long(const uint64_t *__restrict__ key, uint32_t n, uint32_t i, uint64_t top)
{
    constexpr uint32_t H = FIX_LONG_MAX / 2;
    const bool far = (i >= H && (key[i - H] >> LOW_BITS) == top) || (i + H < n && (key[i + H] >> LOW_BITS) == top);
    if (!far) return false;
    uint32_t lo = 0, hi = i;                       // first entry of the run: smallest j with top(j) == top
    while (lo < hi) { const uint32_t mid = lo + (hi - lo) / 2; if ((key[mid] >> LOW_BITS) < top) lo = mid + 1; else hi = mid; }
    const uint32_t first = lo;
    lo = i + 1; hi = n;                            // one past its last entry
    while (lo < hi) { const uint32_t mid = lo + (hi - lo) / 2; if ((key[mid] >> LOW_BITS) <= top) lo = mid + 1; else hi = mid; }
    return lo - first > (uint32_t)FIX_LONG_MAX;
}

// Runs of equal upper bits (key >> LOW_BITS) after the fast passes: inside a run the keys are in ascending original index and
// still have to be ordered by their low bits, stably.  One thread per run start measures the run, up to FIX_LONG_MAX + 1 entries and no
// further; runs that are already in order cost that one scan.  A run too long for the fix-up kernels needs the eight-pass build unless it is
// in order already (coincident particles): that is decided in parallel, by every entry that sees a larger key right before it in its run.
__global__ void __launch_bounds__(SORT_TPB) k_sort_fix_short(uint64_t *__restrict__ key, uint32_t *__restrict__ val, uint32_t n,
                                                              uint2 *__restrict__ long_runs, uint32_t long_cap, uint32_t *__restrict__ n_long,
                                                              uint32_t *__restrict__ flags)
{
    const uint32_t i = blockIdx.x * SORT_TPB + threadIdx.x;
    if (i >= n) return;
    const uint64_t ki = key[i];
    const uint64_t top = ki >> LOW_BITS;
    if (i > 0) {
        const uint64_t kp = key[i - 1];
        if ((kp >> LOW_BITS) == top) {                              // not the first of its run
            // (a short run may be mid-way through its insertion sort here: kp > ki is then unreliable, but such a run is never too long)
            if (kp > ki && *reinterpret_cast<volatile uint32_t *>(flags + 3) == 0u && run_too_long(key, n, i, top)) atomicExch(flags + 3, 1u);
            return;
        }
    }
    if (i + 1 >= n || (key[i + 1] >> LOW_BITS) != top) return;      // a run of one
    uint32_t len = 1;
    bool ordered = true;
    uint64_t prev = ki;
    while (i + len < n && len <= (uint32_t)FIX_LONG_MAX) {
        const uint64_t kj = key[i + len];
        if ((kj >> LOW_BITS) != top) break;
        ordered = ordered && prev <= kj;
        prev = kj;
        len++;
    }
    if (len > (uint32_t)FIX_LONG_MAX) return;                       // too long to fix here; its inversions, if any, raise flags[3] above
    if (ordered) return;
    if (len <= (uint32_t)FIX_SHORT_MAX) {
        for (uint32_t a = 1; a < len; a++) {                       // stable insertion sort: an entry passes strictly larger keys only
            const uint64_t k = key[i + a];
            const uint32_t v = val[i + a];
            uint32_t b = a;
            while (b > 0 && key[i + b - 1] > k) { key[i + b] = key[i + b - 1]; val[i + b] = val[i + b - 1]; b--; }
            key[i + b] = k; val[i + b] = v;
        }
    } else {
        const uint32_t at = atomicAdd(n_long, 1u);
        if (at < long_cap) long_runs[at] = make_uint2(i, len);
        else atomicExch(flags + 3, 1u);
    }
}

// One CTA per long run: rank of an entry = number of entries with a smaller key, or with an equal key and an earlier place.
__global__ void __launch_bounds__(SORT_TPB) k_sort_fix_long(uint64_t *__restrict__ key, uint32_t *__restrict__ val, const uint2 *__restrict__ long_runs,
                                                             uint32_t long_cap, const uint32_t *__restrict__ n_long)
{
    __shared__ uint64_t sk[FIX_LONG_MAX];
    __shared__ uint32_t sv[FIX_LONG_MAX];
    const uint32_t n_runs = min(*n_long, long_cap);
    for (uint32_t r = blockIdx.x; r < n_runs; r += gridDim.x) {
        const uint2 run = long_runs[r];
        for (uint32_t e = threadIdx.x; e < run.y; e += SORT_TPB) { sk[e] = key[run.x + e]; sv[e] = val[run.x + e]; }
        __syncthreads();
        for (uint32_t e = threadIdx.x; e < run.y; e += SORT_TPB) {
            const uint64_t k = sk[e];
            uint32_t rank = 0;
            for (uint32_t j = 0; j < run.y; j++) rank += (sk[j] < k || (sk[j] == k && j < e)) ? 1u : 0u;
            key[run.x + rank] = k;
            val[run.x + rank] = sv[e];
        }
        __syncthreads();
    }
}

} // namespace

static size_t sort_long_cap(uint32_t n_max) { return (size_t)n_max / (FIX_SHORT_MAX + 1) + 1; }

size_t gothic_sort_scratch_bytes(uint32_t n_max)
{
    const size_t ntiles = ((size_t)n_max + TILE - 1) / TILE;
    return (sort_words_head() + (size_t)NPASS * ntiles * RADIX + 2 * sort_long_cap(n_max) + 4) * sizeof(uint32_t);
}

cudaError_t gothic_sort_config()
{
    cudaError_t e = cudaFuncSetAttribute(k_sort_onesweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SortSmem));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_sort_onesweep, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    return e;
}

int gothic_stage_sort(gothic_ctx *c, uint32_t n, bool full, cudaStream_t s)
{
    const uint32_t ntiles = (n + TILE - 1) / TILE, ntiles_max = (c->n_max + TILE - 1) / TILE;
    uint32_t *words = static_cast<uint32_t *>(c->sort_tmp);
    uint32_t *ghist = words, *ticket = words + NPASS * RADIX, *status = words + sort_words_head();
    uint32_t *n_long = status + (size_t)NPASS * ntiles_max * RADIX;
    uint2 *long_runs = reinterpret_cast<uint2 *>(n_long + 4);
    const int npass = full ? NPASS : NPASS_FAST, shift0 = full ? 0 : LOW_BITS;
    GOTHIC_CUDA_OK(c, cudaMemsetAsync(words, 0, (sort_words_head() + (size_t)NPASS * ntiles * RADIX) * sizeof(uint32_t), s));
    int grid = (int)((n + SORT_TPB - 1) / SORT_TPB);
    if (grid > c->num_sms * 8) grid = c->num_sms * 8;
    k_sort_hist<<<grid, SORT_TPB, 0, s>>>(c->key[c->cur], n, ghist, shift0, npass);
    GOTHIC_LAUNCH_OK(c);
    k_sort_scan<<<npass, RADIX, 0, s>>>(ghist);
    GOTHIC_LAUNCH_OK(c);
    for (int p = 0; p < npass; p++) {
        const int in = c->cur, out = c->cur ^ 1;
        k_sort_onesweep<<<ntiles, SORT_TPB, sizeof(SortSmem), s>>>(c->key[in], p == 0 ? nullptr : c->idx[in], c->key[out], c->idx[out], n, shift0 + 8 * p,
                                                                    ghist + p * RADIX, ticket + p, status + (size_t)p * ntiles * RADIX);
        GOTHIC_LAUNCH_OK(c);
        c->cur = out;
    }
    if (!full) {
        GOTHIC_CUDA_OK(c, cudaMemsetAsync(n_long, 0, sizeof(uint32_t), s));
        const uint32_t long_cap = (uint32_t)sort_long_cap(c->n_max);
        k_sort_fix_short<<<(n + SORT_TPB - 1) / SORT_TPB, SORT_TPB, 0, s>>>(c->key[c->cur], c->idx[c->cur], n, long_runs, long_cap, n_long, c->flags);
        GOTHIC_LAUNCH_OK(c);
        k_sort_fix_long<<<c->num_sms * 2, SORT_TPB, 0, s>>>(c->key[c->cur], c->idx[c->cur], long_runs, long_cap, n_long);
        GOTHIC_LAUNCH_OK(c);
    }
    return GOTHIC_OK;
}
