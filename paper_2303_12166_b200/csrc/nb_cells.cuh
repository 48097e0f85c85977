// nb_cells.cuh -- row a3: the contact pairs of Eqs. 5/6 through a
// CELL LIST, rebuilt from scratch at every force evaluation (the result is a function of the state alone,
// so restarts stay bitwise).  Included after nb_kernels.cuh (uses its DevState, ContactArgs, contact_term).
//
// Each star s has its own grid of cubic cells of edge h_s = max(2 R_s, R_0 + R_1): at least the reach of
// any pair that involves an element of s, so a query touches <= 3 cells per axis, and no larger than needed
// for the star with the smaller elements (with the packing of the configs, ~1.2 elements per cell of 2 R:
// the 27 cells of a query hold ~33 candidates for ~5 contacts).  Cell coordinates are counted from the
// star's mean position (robust against a few far outliers) and WRAPPED onto a table of mx x my x mz buckets,
// powers of two >= 4 with at most cap_s (2-4 n_s) buckets: the cells of a query are then distinct buckets,
// x-adjacent cells are adjacent buckets (one range of the sorted array per row of a query), and elements far
// outside the table merely alias onto it (more candidates, same pairs: which pairs ARE in contact is decided
// by contact_term() in fp64).  Containment needs no slack beyond the rounding of R_i + R_j: rounding,
// subtraction of the origin, scaling, floor and clamping are all monotone, so x_i - D <= x_j <= x_i + D puts
// j's cell inside i's range of cells on every axis.
//
//   nb_cell_bbox_kernel     per-star bounding boxes, coordinate sums and counts (block partials); zeroes the counters
//   nb_cell_count_kernel    grid geometry (every block, from the partials); bucket of every element and
//                           its arrival number there (integer atomics: the COUNTS are deterministic)
//   nb_cell_scan_kernel x2  exclusive prefix sum of the counts -> first sorted position of every bucket
//   nb_cell_scatter_kernel  element index -> its bucket's range, in arrival order
//   nb_cell_rank_kernel     ... re-ranked by element index inside the bucket (a fixed order, whatever the
//                           atomics did) and gathered: ps = (x,y,z,R_star), vs = (vx,vy,vz,m)
//   nb_contact_cell_kernel  1 or 4 lanes per element in sorted order: own star's grid, then the other's
//                           (skipped when the element is out of reach of that star's bounding box); fp32
//                           pre-test, survivors queued per lane, the warp's queued pairs dealt evenly to its
//                           lanes and evaluated in fp64, summed per element in the order found
// The seven launches are chained by programmatic dependent launch (pdl_prologue()).
//
// No library code: the sort is a counting sort by bucket written out here.
#pragma once
#include "nb_kernels.cuh"

namespace nb {

constexpr int kCellMinDim = 4;         // >= 3, so that the cells of a query are distinct buckets
constexpr float kCellMaxCoord = 1073741824.f;   // 2^30: cell coordinates are clamped to +-this

struct CellGrid {
    float org[3];          // origin of the cell coordinates: the star's mean position
    float inv_h;           // 1 / cell edge (0: no element, or no reach)
    int mx, my, mz;        // table dimensions - 1 (powers of two)
    int sy, sz;            // log2(dim x), log2(dim x * dim y)
    int base;              // first bucket of this star in the table
    int count;             // elements of this star
    float blo[3], bhi[3];  // bounding box of its elements
};

struct CellState { CellGrid g[2]; };

__device__ __forceinline__ int cell_coord(float x, float org, float inv_h) {
    return __float2int_rd(fminf(fmaxf((x - org) * inv_h, -kCellMaxCoord), kCellMaxCoord));
}
__device__ __forceinline__ int cell_bucket(const CellGrid& g, int ix, int iy, int iz) {
    return g.base + (ix & g.mx) + ((iy & g.my) << g.sy) + ((iz & g.mz) << g.sz);
}

// The kernels of the pass are launched with programmatic stream serialisation (PDL): each lets its successor
// start launching at once and then waits until its predecessor has completed and flushed, so the ~2 us launch
// latency of the seven dependent launches overlaps the kernels instead of separating them.
__device__ __forceinline__ void pdl_prologue() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Block b's grid-stride share of star s: part[2 b + s].
struct CellPartial { float lo[3]; int cnt; float hi[3]; float pad0; float sum[3]; float pad1; };

constexpr int kPassThreads = 256;      // threads per block of the pass
constexpr int kPassMaxBlocks = 1024;   // most blocks (= partial boxes) of the pass
constexpr int kCellScanChunk = 4 * kPassThreads;   // counters per block-wide scan

struct CellPassArgs {
    const float4* __restrict__ posm;
    const float4* __restrict__ vel;
    const DevState* __restrict__ dev;
    CellPartial* __restrict__ part;    // [2 * blocks]
    CellState* __restrict__ cs;
    int* __restrict__ counters;        // [ncells + 1]: counts, then first sorted positions
    int* __restrict__ bsum;            // [ceil(ncells / kCellScanChunk)] chunk sums, then their prefix
    int* __restrict__ bucket;          // [n] bucket of element i
    int* __restrict__ slot;            // [n] its arrival number there
    int* __restrict__ tmp;             // [n] element indices by bucket, arrival order
    uint32_t* __restrict__ perm;       // [n] element indices by bucket, index order
    float4* __restrict__ ps;           // [n] x,y,z,R_star   (sorted by star, bucket, index)
    float4* __restrict__ vs;           // [n] vx,vy,vz,m
    float4* __restrict__ out;          // [n] contact acceleration, ORIGINAL index order
    double* __restrict__ epart;        // energy mode (nb_energy): U_rep of the block's pairs, one fp64 partial per block
    unsigned long long* __restrict__ stats;   // counting mode (nb_contact_stats): candidates pre-tested, pairs queued
    ContactArgs law;                   // gamma, gamma_beta, v_dead, lens_mode
    int n, n1, cap0, cap1, ncells;     // cap_s: buckets of star s (0 or a power of two >= 64); ncells = cap0 + cap1
    int lpe_log2;                      // lanes per element of the contact phase: 1 << lpe_log2 <= 32
    int nparts;                        // blocks of the bbox phase (= partial boxes)
};

// Inclusive scan of one int per thread over the block (kPassThreads threads); *total = the block's sum.
__device__ __forceinline__ int block_scan_inclusive(int v, int* sh /*[8]*/, int* total)
{
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, v, o); if (l >= o) v += t; }
    __syncthreads();                                          // sh may still be read from the previous call
    if (l == 31) sh[w] = v;
    __syncthreads();
    int before = 0, tot = 0;
#pragma unroll
    for (int k = 0; k < kPassThreads / 32; ++k) { const int t = sh[k]; if (k < w) before += t; tot += t; }
    *total = tot;
    return v + before;
}

// Phase 0: per-star bounding boxes, coordinate sums and counts of this block's share; counters zeroed.
__device__ __forceinline__ void cell_phase_bbox(const CellPassArgs& a)
{
    __shared__ float sh[2][9][kPassThreads / 32];
    __shared__ int shc[2][kPassThreads / 32];
    const int gt = blockIdx.x * kPassThreads + threadIdx.x, stride = gridDim.x * kPassThreads;
    for (int c = gt; c <= a.ncells; c += stride) a.counters[c] = 0;
    float q[2][9];
    int cnt[2] = {0, 0};
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int c = 0; c < 3; ++c) { q[s][c] = 3.0e38f; q[s][3 + c] = -3.0e38f; q[s][6 + c] = 0.f; }
    for (int i = gt; i < a.n; i += stride) {
        const float4 p = a.posm[i];
        const float x[3] = {p.x, p.y, p.z};
        const bool first = i < a.n1;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            if ((s == 0) == first) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    q[s][c] = fminf(q[s][c], x[c]); q[s][3 + c] = fmaxf(q[s][3 + c], x[c]); q[s][6 + c] += x[c];
                }
                ++cnt[s];
            }
        }
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
#pragma unroll
    for (int s = 0; s < 2; ++s) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float lo = warp_min(q[s][c]), hi = warp_max(q[s][3 + c]);
            float t = q[s][6 + c];
            for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
            if (l == 0) { sh[s][c][w] = lo; sh[s][3 + c][w] = hi; sh[s][6 + c][w] = t; }
        }
        int k = cnt[s];
        for (int o = 16; o > 0; o >>= 1) k += __shfl_xor_sync(0xffffffffu, k, o);
        if (l == 0) shc[s][w] = k;
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        const int s = threadIdx.x;
        CellPartial r;
        for (int c = 0; c < 3; ++c) {
            float lo = sh[s][c][0], hi = sh[s][3 + c][0], t = sh[s][6 + c][0];
            for (int k = 1; k < kPassThreads / 32; ++k) {
                lo = fminf(lo, sh[s][c][k]); hi = fmaxf(hi, sh[s][3 + c][k]); t += sh[s][6 + c][k];
            }
            r.lo[c] = lo; r.hi[c] = hi; r.sum[c] = t;
        }
        int k = 0;
        for (int j = 0; j < kPassThreads / 32; ++j) k += shc[s][j];
        r.cnt = k; r.pad0 = r.pad1 = 0.f;
        a.part[2 * blockIdx.x + s] = r;
    }
}

// Geometry of star s's grid from the blocks' partials.  Called by one full warp; the result is the same
// in every lane (xor butterflies) and in every block (same inputs, same order).
__device__ __forceinline__ CellGrid cell_make_grid(const CellPartial* __restrict__ part, int nparts, int s, float R0,
                                                   float R1, int base, int cap)
{
    const int l = threadIdx.x & 31;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, sum[3] = {0.f, 0.f, 0.f};
    int cnt = 0;
    for (int b = l; b < nparts; b += 32) {
        const CellPartial q = part[2 * b + s];
#pragma unroll
        for (int c = 0; c < 3; ++c) { lo[c] = fminf(lo[c], q.lo[c]); hi[c] = fmaxf(hi[c], q.hi[c]); sum[c] += q.sum[c]; }
        cnt += q.cnt;
    }
    for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    CellGrid g;
    const float h = fmaxf(2.f * (s ? R1 : R0), R0 + R1) * (1.f + 1.0e-5f);
    g.inv_h = (h > 0.f && cnt > 0) ? 1.f / h : 0.f;
    float need[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        lo[c] = warp_min(lo[c]); hi[c] = warp_max(hi[c]);
        float t = sum[c];
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        g.org[c] = cnt > 0 ? t / (float)cnt : 0.f;
        g.blo[c] = lo[c]; g.bhi[c] = hi[c];
        need[c] = cnt > 0 ? fminf((hi[c] - lo[c]) * g.inv_h + 2.f, 1.0e6f) : 1.f;
        if (!(need[c] >= 1.f)) need[c] = 1.f;                    // NaN positions: any grid will do
    }
    int m[3] = {kCellMinDim, kCellMinDim, kCellMinDim};
#pragma unroll
    for (int c = 0; c < 3; ++c) while ((float)m[c] < need[c]) m[c] <<= 1;
    while ((long long)m[0] * m[1] * m[2] > (long long)(cap > 64 ? cap : 64)) {   // too many buckets: wrap the longest axis
        int c = 0;
        if (m[1] > m[c]) c = 1;
        if (m[2] > m[c]) c = 2;
        m[c] >>= 1;
    }
    if (!(g.inv_h > 0.f)) {                                      // no reach (every radius 0 at this step): nobody will query
        m[1] = m[2] = kCellMinDim;                               // this grid; the elements are dealt over all its buckets
        m[0] = (cap > 64 ? cap : 64) / (kCellMinDim * kCellMinDim);   // by index (cell_phase_count), not piled into one
    }
    g.mx = m[0] - 1; g.my = m[1] - 1; g.mz = m[2] - 1;
    g.sy = 31 - __clz(m[0]); g.sz = g.sy + 31 - __clz(m[1]);
    g.base = base; g.count = cnt;
    return g;
}

// Phase 1: the grids (every block, from the partials); bucket and arrival number of every element.
__device__ __forceinline__ void cell_phase_count(const CellPassArgs& a, CellGrid* sg /*shared [2]*/)
{
    const int w = threadIdx.x >> 5;
    if (w < 2) {
        const float R0 = a.dev->R[0], R1 = a.dev->R[1];
        const CellGrid g = cell_make_grid(a.part, a.nparts, w, R0, R1, w ? a.cap0 : 0, w ? a.cap1 : a.cap0);
        if ((threadIdx.x & 31) == 0) {
            sg[w] = g;
            if (blockIdx.x == 0) a.cs->g[w] = g;
        }
    }
    __syncthreads();
    for (int i = blockIdx.x * kPassThreads + threadIdx.x; i < a.n; i += gridDim.x * kPassThreads) {
        const float4 p = a.posm[i];
        const CellGrid& g = sg[i < a.n1 ? 0 : 1];
        int b;
        if (g.inv_h > 0.f)
            b = cell_bucket(g, cell_coord(p.x, g.org[0], g.inv_h), cell_coord(p.y, g.org[1], g.inv_h),
                            cell_coord(p.z, g.org[2], g.inv_h));
        else                                                     // a grid without reach: one element per bucket, by index
            b = g.base + ((i < a.n1 ? i : i - a.n1) & ((g.mx + 1) * (g.my + 1) * (g.mz + 1) - 1));   // (a power of two >= 2 n_s)
        a.bucket[i] = b;
        a.slot[i] = atomicAdd(&a.counters[b], 1);
    }
}

// Phases 2a-2c: exclusive prefix sum of counters[0..ncells) in place, counters[ncells] = n.
//   phase 0: bsum[chunk] = sum of the chunk;  phase 1: block 0 turns bsum into its exclusive prefix;
//   phase 2: every chunk scanned on top of bsum[chunk];  phase 3 = phase 2 without phase 1 before it (every block
//   adds up the chunk sums before its own).
__device__ __forceinline__ void cell_phase_scan(const CellPassArgs& a, int phase, int* sh /*shared [8]*/)
{
    const int nchunks = (a.ncells + kCellScanChunk - 1) / kCellScanChunk;
    if (phase == 1) {                         // block 0: exclusive prefix of the chunk sums
        if (blockIdx.x != 0) return;
        int carry = 0;
        for (int c0 = 0; c0 < nchunks; c0 += kPassThreads) {
            const int c = c0 + threadIdx.x;
            const int v = c < nchunks ? a.bsum[c] : 0;
            int tot;
            const int inc = block_scan_inclusive(v, sh, &tot);
            if (c < nchunks) a.bsum[c] = carry + inc - v;
            carry += tot;
        }
        return;
    }
    for (int ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
        const int c0 = ch * kCellScanChunk + threadIdx.x * 4;
        int v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = (c0 + k < a.ncells) ? a.counters[c0 + k] : 0;
        const int mine = v[0] + v[1] + v[2] + v[3];
        int tot;
        const int inc = block_scan_inclusive(mine, sh, &tot);
        if (phase == 0) {
            if (threadIdx.x == 0) a.bsum[ch] = tot;
        } else {
            int base;
            if (phase == 2) base = a.bsum[ch];
            else {
                int t = 0;
                for (int b = threadIdx.x; b < ch; b += kPassThreads) t += a.bsum[b];
                int dummy;
                base = block_scan_inclusive(t, sh, &dummy);
                base = dummy;
            }
            int e = base + inc - mine;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (c0 + k < a.ncells) a.counters[c0 + k] = e;
                e += v[k];
            }
            if (c0 <= a.ncells - 1 && a.ncells - 1 < c0 + 4) a.counters[a.ncells] = e;
        }
    }
}

// Phase 3: element index -> its bucket's range of sorted positions, in arrival order.
__device__ __forceinline__ void cell_phase_scatter(const CellPassArgs& a)
{
    for (int i = blockIdx.x * kPassThreads + threadIdx.x; i < a.n; i += gridDim.x * kPassThreads)
        a.tmp[a.counters[a.bucket[i]] + a.slot[i]] = i;
}

// Phase 4: sorted position p holds, in arrival order, some element of bucket b; its final place is the number
// of elements of b with a smaller index -- a fixed order, whatever the atomics did.  Buckets hold ~1 element
// (all of a star only when the whole star fits into one cell, and then every pair is a candidate anyway).
__device__ __forceinline__ void cell_phase_rank(const CellPassArgs& a)
{
    const float R0 = a.dev->R[0], R1 = a.dev->R[1];
    for (int p = blockIdx.x * kPassThreads + threadIdx.x; p < a.n; p += gridDim.x * kPassThreads) {
        const int idx = a.tmp[p];
        const int b = a.bucket[idx];
        const int s0 = a.counters[b], s1 = a.counters[b + 1];
        int rank = 0;
        for (int q = s0; q < s1; ++q) rank += (a.tmp[q] < idx);
        const int dst = s0 + rank;
        const float4 x = a.posm[idx], v = a.vel[idx];
        a.perm[dst] = (uint32_t)idx;
        a.ps[dst] = make_float4(x.x, x.y, x.z, star_radius(idx, a.n1, R0, R1));
        a.vs[dst] = make_float4(v.x, v.y, v.z, x.w);
    }
}

constexpr int kCcThreads = 128;        // threads per block of the contact kernel
constexpr int kCcQueue = 16;           // per-lane queue of pairs that passed the fp32 pre-test
constexpr int kCcRound = 64;           // pairs a warp evaluates per round of the balanced evaluation

// Eqs. 5/6 over the cell list.  2^LPL lanes share one element: lane q takes the rows q, q + LPE, ... of the
// element's query (a row = the x-run of cells at one (y, z): one range of sorted positions, two if it wraps),
// own star's grid first, then the other's.
//   1. the ranges of the lane's rows are fetched together (one memory latency, not one per row) and walked
//      as ONE loop over candidates, so a warp takes as long as its busiest lane, not the sum of the busiest
//      lane of every row;
//   2. pairs that pass the fp32 pre-test wait in the lane's queue (if it overflows -- dense overlaps -- the
//      lane evaluates it on the spot);
//   3. the queued pairs of the whole warp are dealt evenly to its lanes (a lane with 11 contacts no longer
//      holds up 31 lanes with 4), evaluated in fp64 and handed back through shared memory; every lane adds
//      up ITS pairs in the order it found them, and the lanes of an element are added by a fixed shuffle tree:
//      the sums are bitwise reproducible.
// ENERGY = true (nb_energy, row a7): the same search, but every queued pair (k, j) with k < j in sorted order adds its
// repulsion potential U_rep (reading A12) to one fp64 partial per block instead of a force to element k.
// STATS = true (nb_contact_stats, a measurement aid): also counts the candidates it pre-tests and the pairs it queues.
template <int LPL, bool ENERGY = false, bool STATS = false>
__global__ void __launch_bounds__(kCcThreads)
nb_contact_cell_kernel(const __grid_constant__ CellPassArgs a)
{
    constexpr int LPE = 1 << LPL;
    constexpr int ROWS = (9 + LPE - 1) / LPE;      // rows of a 3 x 3 query per lane
    constexpr int RC = 2 * ROWS;                   // ranges per lane and batch
    __shared__ CellGrid sg[2];
    __shared__ int rng[RC][2][kCcThreads];
    __shared__ uint32_t hq[kCcQueue + 1][kCcThreads];
    __shared__ int pre[kCcThreads / 32][33];
    __shared__ double invm[kCcThreads];
    __shared__ double res[kCcThreads / 32][kCcRound][3];
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    pdl_prologue();
    if (tid < 2) sg[tid] = a.cs->g[tid];
    __syncthreads();
    const int q = lane & (LPE - 1);
    const float kSlack = 1.0f + 1.0e-5f;           // the fp32 test is a pre-filter; contact_pair() decides in fp64
    const float R[2] = {a.dev->R[0], a.dev->R[1]};
    const int n0 = sg[0].count;
    const long long base = (long long)blockIdx.x * kCcThreads + (tid & ~31);     // first item of this warp
    const int k = (int)((base + lane) >> LPL);
    const bool valid = k < a.n;
    double ax = 0.0, ay = 0.0, az = 0.0;
    int nh = 0;
    unsigned ncand = 0, nqueued = 0;
    float4 pi = make_float4(0.f, 0.f, 0.f, 0.f), vi = make_float4(0.f, 0.f, 0.f, 1.f);
    if (valid) {
        pi = a.ps[k]; vi = a.vs[k];
        const int si = k < n0 ? 0 : 1;
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            const int t = pass ? 1 - si : si;
            const CellGrid& g = sg[t];
            if (g.count == 0 || !(g.inv_h > 0.f)) continue;
            const float Dx = pi.w + R[t];
            const float D = Dx * (1.0f + 1.0e-6f);                   // >= R_i + R_j exactly
            if (!(D > 0.f)) continue;
            if (pass) {                             // out of reach of the other star's bounding box: nothing there
                const float gx = fmaxf(0.f, fmaxf(g.blo[0] - pi.x, pi.x - g.bhi[0]));
                const float gy = fmaxf(0.f, fmaxf(g.blo[1] - pi.y, pi.y - g.bhi[1]));
                const float gz = fmaxf(0.f, fmaxf(g.blo[2] - pi.z, pi.z - g.bhi[2]));
                if (gx * gx + gy * gy + gz * gz > D * D * kSlack) continue;
            }
            const float thr = Dx * Dx * kSlack;
            const int x0 = cell_coord(pi.x - D, g.org[0], g.inv_h), x1 = cell_coord(pi.x + D, g.org[0], g.inv_h);
            const int y0 = cell_coord(pi.y - D, g.org[1], g.inv_h), y1 = cell_coord(pi.y + D, g.org[1], g.inv_h);
            const int z0 = cell_coord(pi.z - D, g.org[2], g.inv_h), z1 = cell_coord(pi.z + D, g.org[2], g.inv_h);
            const int nx = min(x1 - x0, g.mx) + 1, ny = min(y1 - y0, g.my) + 1, nz = min(z1 - z0, g.mz) + 1;
            const int c0 = x0 & g.mx;
            const int run0 = min(nx, g.mx + 1 - c0);                 // cells before the table wraps in x
            const int nrows = ny * nz;
            const int* __restrict__ start = a.counters;
            const float4* __restrict__ psj = a.ps;
#pragma unroll 1
            for (int r0 = 0; r0 < nrows; r0 += ROWS * LPE) {
                int nr = 0;
#pragma unroll
                for (int u = 0; u < ROWS; ++u) {                     // the ranges of this batch of rows, fetched together
                    const int r = r0 + q + u * LPE;
                    if (r < nrows) {
                        int rz;
                        if (nrows <= 9) rz = (r >= ny) + (r >= 2 * ny) + (r >= 3 * ny) + (r >= 4 * ny) + (r >= 5 * ny)
                                           + (r >= 6 * ny) + (r >= 7 * ny) + (r >= 8 * ny);      // r / ny without the division
                        else rz = r / ny;
                        const int ry = r - rz * ny;
                        const int row = g.base + (((y0 + ry) & g.my) << g.sy) + (((z0 + rz) & g.mz) << g.sz);
                        const int j0 = start[row + c0], j1 = start[row + c0 + run0];
                        rng[nr][0][tid] = j0; rng[nr][1][tid] = j1;
                        nr += (j1 > j0);
                        if (run0 < nx) {                             // the run wrapped: the rest starts at x = 0
                            const int k0 = start[row], k1 = start[row + nx - run0];
                            rng[nr][0][tid] = k0; rng[nr][1][tid] = k1;
                            nr += (k1 > k0);
                        }
                    }
                }
                int ri = 0, j = 0, je = 0;
                while (true) {                                       // one loop over all candidates of the batch
                    if (j == je) {
                        if (ri == nr) break;
                        j = rng[ri][0][tid]; je = rng[ri][1][tid]; ++ri;
                    }
                    const float4 pj = psj[j];
                    const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
                    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    hq[nh][tid] = (uint32_t)j;                       // kept only if it is a hit
                    nh += (r2 <= thr && j != k);
                    if (STATS) { ++ncand; nqueued += (r2 <= thr && j != k); }
                    ++j;
                    if (nh == kCcQueue) {                            // queue full (dense overlaps): evaluate it here, in order
                        const double im = 1.0 / (double)vi.w;
                        for (int h = 0; h < nh; ++h) {
                            const int jj = (int)hq[h][tid];
                            double fx, fy, fz;
                            if (ENERGY) { if (k < jj) ax += contact_potential(a.law, pi, a.ps[jj]); continue; }
                            contact_pair(a.law, pi, vi, a.ps[jj], a.vs[jj], fx, fy, fz);
                            ax += fx * im; ay += fy * im; az += fz * im;
                        }
                        nh = 0;
                    }
                }
            }
        }
    }
    if (STATS) {
        for (int o = 16; o > 0; o >>= 1) { ncand += __shfl_xor_sync(0xffffffffu, ncand, o); nqueued += __shfl_xor_sync(0xffffffffu, nqueued, o); }
        if (lane == 0) { atomicAdd(a.stats, (unsigned long long)ncand); atomicAdd(a.stats + 1, (unsigned long long)nqueued); }
    }
    // balanced evaluation of the warp's queued pairs
    __syncwarp();
    int inc = nh;
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    const int total = __shfl_sync(0xffffffffu, inc, 31);
    const int mine0 = inc - nh;
    pre[w][lane] = mine0;
    if (lane == 31) pre[w][32] = total;
    invm[tid] = 1.0 / (double)vi.w;
    __syncwarp();
    const double im = invm[tid];
    for (int p0 = 0; p0 < total; p0 += kCcRound) {
        const int pe = min(total, p0 + kCcRound);
        for (int p = p0 + lane; p < pe; p += 32) {
            int lo = 0;                              // owner: the largest lane with pre[lane] <= p
#pragma unroll
            for (int s2 = 16; s2 > 0; s2 >>= 1) if (pre[w][lo + s2] <= p) lo += s2;
            const int ot = (tid & ~31) + lo;
            const int jj = (int)hq[p - pre[w][lo]][ot];
            const int ko = (int)((base + lo) >> LPL);
            double fx, fy = 0.0, fz = 0.0;
            if (ENERGY) fx = ko < jj ? contact_potential(a.law, a.ps[ko], a.ps[jj]) : 0.0;
            else contact_pair(a.law, a.ps[ko], a.vs[ko], a.ps[jj], a.vs[jj], fx, fy, fz);
            res[w][p - p0][0] = fx; res[w][p - p0][1] = fy; res[w][p - p0][2] = fz;
        }
        __syncwarp();
        const int b = max(mine0, p0), e = min(mine0 + nh, pe);
        for (int p = b; p < e; ++p) {
            if (ENERGY) { ax += res[w][p - p0][0]; continue; }
            ax += res[w][p - p0][0] * im; ay += res[w][p - p0][1] * im; az += res[w][p - p0][2] * im;
        }
        __syncwarp();
    }
#pragma unroll
    for (int o = LPE >> 1; o > 0; o >>= 1) {        // lanes q + o -> q: a fixed tree
        ax += __shfl_down_sync(0xffffffffu, ax, o);
        ay += __shfl_down_sync(0xffffffffu, ay, o);
        az += __shfl_down_sync(0xffffffffu, az, o);
    }
    if (ENERGY) {                                    // lane 0 of every element group holds the group's sum: add up the block's
        __shared__ double esum[kCcThreads / 32];
        double v = (valid && q == 0) ? ax : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) esum[w] = v;
        __syncthreads();
        if (tid == 0) {
            double t = 0.0;
            for (int i = 0; i < kCcThreads / 32; ++i) t += esum[i];
            a.epart[blockIdx.x] = t;
        }
        return;
    }
    if (valid && q == 0) a.out[a.perm[k]] = make_float4((float)ax, (float)ay, (float)az, 0.f);
}

// Phases 0-4 as kernels.
__global__ void __launch_bounds__(kPassThreads) nb_cell_bbox_kernel(const __grid_constant__ CellPassArgs a)
{
    pdl_prologue();
    cell_phase_bbox(a);
}
__global__ void __launch_bounds__(kPassThreads) nb_cell_count_kernel(const __grid_constant__ CellPassArgs a)
{
    __shared__ CellGrid sg[2];
    pdl_prologue();
    cell_phase_count(a, sg);
}
__global__ void __launch_bounds__(kPassThreads) nb_cell_scan_kernel(const __grid_constant__ CellPassArgs a, int phase)
{
    __shared__ int sh_scan[kPassThreads / 32];
    pdl_prologue();
    cell_phase_scan(a, phase, sh_scan);
}
__global__ void __launch_bounds__(kPassThreads) nb_cell_scatter_kernel(const __grid_constant__ CellPassArgs a)
{
    pdl_prologue();
    cell_phase_scatter(a);
}
__global__ void __launch_bounds__(kPassThreads) nb_cell_rank_kernel(const __grid_constant__ CellPassArgs a)
{
    pdl_prologue();
    cell_phase_rank(a);
}

}  // namespace nb
