// nb_api.cu -- host side of the C ABI declared in include/nb.h.
// Argument validation, launch configuration and kernel sequencing only; every
// arithmetic step of the path runs in the kernels of nb_kernels.cuh.
#include "nb.h"
#include "nb_kernels.cuh"
#include "nb_cells.cuh"
#include "nb_fused.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

using namespace nb;

namespace {

constexpr int64_t kMaxN = (int64_t)1 << 26;       // 67M elements: int indexing, n*TJ fits
constexpr int kNumSMsFallback = 148;
constexpr int kMomentBlocks = 296;
constexpr size_t kAlign = 256;

inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Plan {           // launch configuration of the gravity kernel for a given n
    int I = 2;          // elements i per thread
    int TJ = 256;       // j tile
    int nib = 0;        // i blocks
    int njt = 0;        // j tiles
    int nsplit = 1;     // j splits P
    int sym_S = 0;      // > 0: symmetric kernel with super-tiles of sym_S elements (else the one-sided kernel)
    int T = 0;          // symmetric kernel: number of super-tiles = slabs of partial sums
    bool chain = false; // symmetric kernel in chain mode: two fp64 accumulators per element instead of the T slabs
};

constexpr int kCtasPerSM = 8;                      // resident CTAs/SM of nb_gravity_kernel<2, .> (64 registers)
constexpr int64_t kMaxSplit = 64;
constexpr int64_t kPartialBudget = (int64_t)128 << 20;   // bytes of split-j partial sums worth keeping in L2
constexpr int64_t kCellMinN = 8192;                // from here on the contact pass builds the cell list.  Below, contact terms are
                                                   // found inside nb_fused_step_kernel's all-pairs loop; the separate index-order
                                                   // pass (all pairs pre-tested) runs only when that kernel is unavailable or a
                                                   // path is forced, and under nb_time_contact_pass / nb_contact_stats
constexpr int64_t kContactWideN = 131072;          // cell list: below this, 4 lanes share the rows of an element's query
                                                   // (measured: 16,384: 45 vs 67 us per pass, 65,536: 50 vs 53; 262,144: 129 vs 107)
constexpr int kMaxContactChunks = 32;              // index-order search: the candidate groups of a warp go to this many slabs

// Force-path selection (nb_set_force_path).
enum { kPathAuto = 0, kPathOneSided = 1, kPathSymmetric = 2 };
constexpr int64_t kSymMinN = 8192;                // auto: symmetric kernel from here on (below: the fused one-launch kernel).
                                                  // Measured whole steps, one-sided / symmetric, us (profiles/r2_crossover.md):
                                                  // 8,192: 74 / 60, 10,240: 84 / 70, 12,288: 109 / 89, 16,384: 158 / 131,
                                                  // 24,576: 328 / 252
constexpr int64_t kSym256MaxN = 32768;             // below this the super-tiles are 256 elements (CTAs of 2 warps)
constexpr int64_t kSymMaxN = (int64_t)1 << 26;    // ... for every n the library takes
constexpr int64_t kChainMinN = 98304;             // from here on (S >= 1,024) the symmetric kernel runs in chain mode: its T
                                                  // slabs would be 1.1 GB at 262,144 elements and 5 GB at 1,048,576.  Not below:
                                                  // with the short CTAs of S = 512 the turns do cost (65,536: 1.66 vs 1.20 ms)

// Super-tile size of the symmetric kernel for n elements: its T = ceil(n/S) slabs of n float4
// partial sums cost memory and one extra pass, so S grows with n.
int sym_tile(int64_t n)
{
    if (n < kSym256MaxN) return 256;  // small n: more, smaller CTAs (T <= 128)
    if (n < 98304) return 512;        // T <= 192
    if (n < 393216) return 1024;      // T <= 384
    if (n < 786432) return 2048;
    return 4096;                      // (chain mode keeps no slabs; measured at 1,048,576: S = 2,048 299.3 ms, 4,096 299.0)
}

int64_t sym_slabs(int64_t n) { const int64_t S = sym_tile(n); return (n + S - 1) / S; }

// Slabs the contact pass writes for n elements: one (cell list), or one per chunk of candidate groups
// (index-order search, n < kCellMinN).
int contact_slabs(int64_t n)
{
    if (n >= kCellMinN) return 1;
    const int64_t ngroups = (n + kGroup - 1) / kGroup;
    return (int)(ngroups < kMaxContactChunks ? ngroups : kMaxContactChunks);
}

// Buckets of the cell table of a star of ns elements: a power of two in [2 ns, 4 ns), at least 64 (4 x 4 x 4).
int64_t cell_cap(int64_t ns)
{
    if (ns <= 0) return 0;
    int64_t c = 64;
    while (c < 2 * ns) c <<= 1;
    return c;
}

// Largest number of j splits allowed for n elements (bounds the partial-sum slabs).
int64_t max_split(int64_t n)
{
    int64_t p = kPartialBudget / (16 * n);
    if (p < 8) p = 8;
    if (p > kMaxSplit) p = kMaxSplit;
    return p;
}

// Slabs of n float4: max_split(n) gravity partials + 1 contact slab.  Each term of the bound
// grows with n, so the value for n_max covers every n <= n_max.
int64_t partial_elems_bound(int64_t n_max)
{
    const int64_t a = (kMaxSplit + kMaxContactChunks) * n_max;
    const int64_t b1 = 9 * n_max, b2 = kPartialBudget / 16 + n_max;
    const int64_t b = b1 > b2 ? b1 : b2;
    int64_t r = a < b ? a : b;
    // symmetric kernel: (T(n) + 1) n, largest just below each change of the super-tile size
    // (only below kChainMinN: chain mode keeps two fp64 sums per element instead)
    const int64_t top = n_max < kChainMinN - 1 ? n_max : kChainMinN - 1;
    const int64_t tops[1] = {kSym256MaxN - 1};
    int64_t probes[2] = {top, top};
    for (int k = 0; k < 1; ++k) if (tops[k] < top) probes[k + 1] = tops[k];
    for (int64_t n : probes) {
        const int64_t e = (sym_slabs(n) + contact_slabs(n)) * n;
        if (e > r) r = e;
    }
    return r;
}

// P j-splits give nib*P equal CTAs that run in rounds of `slots` resident CTAs: the cost is
// rounds x (tiles per split + a per-CTA prologue), with a small term for the ragged end of
// the last round (CTAs drift apart, so more rounds end more evenly).
Plan make_plan(int64_t n, int num_sms, int path)
{
    Plan p;
    if ((path == kPathSymmetric || (path == kPathAuto && n >= kSymMinN)) && n <= kSymMaxN) {
        p.sym_S = sym_tile(n);
        p.T = (int)sym_slabs(n);
        p.chain = n >= kChainMinN;
    }
    p.I = 2;
    p.TJ = n >= 16384 ? 256 : 128;
    const int ib = kThreads * p.I;
    p.nib = (int)((n + ib - 1) / ib);
    p.njt = (int)((n + p.TJ - 1) / p.TJ);
    const int64_t slots = (int64_t)num_sms * kCtasPerSM;
    int64_t pmax = p.njt >= 2 ? p.njt / 2 : 1;
    if (n < kCellMinN) pmax = p.njt;                 // small n, reached only without the fused kernel (no cooperative launch) and by
                                                     // nb_gravity_accel_static / nb_time_force_kernel: down to one tile per CTA
    if (pmax > max_split(n)) pmax = max_split(n);
    double best = 0.0;
    for (int64_t P = 1; P <= pmax; ++P) {
        const int64_t rounds = (p.nib * P + slots - 1) / slots;
        const int64_t tiles = (p.njt + P - 1) / P;
        const double cost = (double)rounds * (double)(tiles + 2) * (1.0 + 0.25 / (double)rounds);
        if (P == 1 || cost < best) { best = cost; p.nsplit = (int)P; }
    }
    return p;
}

struct Layout {
    size_t off_dev, off_acc, off_part, off_red, off_ps, off_vs, off_gbox, off_sbox, off_cpart, off_cstate,
        off_counters, off_bsum, off_bucket, off_slot, off_tmp, off_perm, off_acc64, off_turn, off_epot, off_erep, off_tbox, off_xfer, total;
};

// Super-tile of nb_pot_pair_kernel for n elements (T <= 512 up to 2M elements), and its CTAs = fp64 partials.
int pot_tile(int64_t n) { return n <= 524288 ? 1024 : (n <= 2097152 ? 4096 : 8192); }
int64_t pot_pairs(int64_t n) { const int64_t T = (n + pot_tile(n) - 1) / pot_tile(n); return T * (T + 1) / 2; }

// cell_cap(n1) + cell_cap(n - n1) < 4 n + 128 for every split of n <= n_max elements
int64_t cell_counters_bound(int64_t n_max) { return 4 * n_max + 129; }

Layout make_layout(int64_t n_max)
{
    Layout L;
    size_t o = 0;
    const size_t ngroups = (size_t)((n_max + kGroup - 1) / kGroup);
    const size_t nsuper = (ngroups + kSuper - 1) / kSuper;
    L.off_dev = o;  o += align_up(sizeof(DevState));
    L.off_acc = o;  o += align_up((size_t)n_max * sizeof(float4));
    L.off_part = o; o += align_up((size_t)partial_elems_bound(n_max) * sizeof(float4));
    const size_t pot_blocks = (size_t)((n_max + kThreads - 1) / kThreads);
    const size_t red = (size_t)kMomentBlocks * 16 * sizeof(double) + pot_blocks * 2 * sizeof(double);   // 16 >= kMomentCols, kXferCols1, kXferCols2
    L.off_red = o;  o += align_up(red);
    L.off_ps = o;   o += align_up((size_t)n_max * sizeof(float4));
    L.off_vs = o;   o += align_up((size_t)n_max * sizeof(float4));
    L.off_gbox = o; o += align_up(ngroups * 2 * sizeof(float4));
    L.off_sbox = o; o += align_up(nsuper * 2 * sizeof(float4));
    const size_t ncnt = (size_t)cell_counters_bound(n_max);
    L.off_cpart = o;    o += align_up((size_t)kPassMaxBlocks * 2 * sizeof(CellPartial));
    L.off_cstate = o;   o += align_up(sizeof(CellState));
    L.off_counters = o; o += align_up(ncnt * sizeof(int));
    L.off_bsum = o;     o += align_up((ncnt / kCellScanChunk + 2) * sizeof(int));
    L.off_bucket = o;   o += align_up((size_t)n_max * sizeof(int));
    L.off_slot = o;     o += align_up((size_t)n_max * sizeof(int));
    L.off_tmp = o;      o += align_up((size_t)n_max * sizeof(int));
    L.off_perm = o;     o += align_up((size_t)n_max * sizeof(uint32_t));
    L.off_acc64 = o;    o += align_up(n_max >= kChainMinN ? (size_t)n_max * 6 * sizeof(double) : 0);
    L.off_turn = o;     o += align_up(n_max >= kChainMinN ? ((size_t)(n_max / 1024 + 1) * 5 + 2) * sizeof(int) : 0);   // <= 4 rounds + 1 per tile
    L.off_epot = o;     o += align_up((size_t)pot_pairs(n_max) * sizeof(double));
    L.off_erep = o;     o += align_up(((size_t)n_max * 4 / kCcThreads + 1) * sizeof(double));
    L.off_tbox = o;     o += align_up(((size_t)n_max / 1024 + 1) * 2 * sizeof(float4));   // nb_energy: boxes of its super-tiles (S >= 1,024)
    L.off_xfer = o;     o += align_up(sizeof(XferGeom)) + align_up(32 * sizeof(double));   // f3: geometry between the passes, and the record of nb_transfer_diagnostics
    L.total = o;
    return L;
}

}  // namespace

struct nb_ctx {
    nb_params prm;
    int64_t n_max = 0, n = 0;
    int n1 = 0;
    cudaStream_t stream = nullptr;
    cudaStream_t side = nullptr;          // library-owned: the contact pass runs here, beside the gravity kernel
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int num_sms = kNumSMsFallback;
    int device = -1;                      // the device that was current at nb_create(): every pointer and kernel attribute belongs to it
    bool fused_ok = false;                // cooperative launch + the shared memory of nb_fused_step_kernel are available
    int fused_blocks = 0, fused_logP = 0; // CTAs of nb_fused_step_kernel for the bound state (0: not available) and its 2^logP pairs per CTA
    float4* posm = nullptr;
    float4* vel = nullptr;
    char* ws = nullptr;
    Layout lay{};
    Plan plan{};
    bool have_state = false, have_acc = false;
    bool acc_uploaded = false;            // the cached a(x) came from nb_upload_state(host_acc), not from a force evaluation here
    bool chain_launched = false;          // the turn counters / error flag of chain mode hold a launch's state
    int path = kPathAuto;
    int last_cuda = 0;
    int64_t launches = 0;

    DevState* dev() const { return reinterpret_cast<DevState*>(ws + lay.off_dev); }
    float4* acc() const { return reinterpret_cast<float4*>(ws + lay.off_acc); }
    float4* part() const { return reinterpret_cast<float4*>(ws + lay.off_part); }
    double* red() const { return reinterpret_cast<double*>(ws + lay.off_red); }
    float4* ps() const { return reinterpret_cast<float4*>(ws + lay.off_ps); }
    float4* vs() const { return reinterpret_cast<float4*>(ws + lay.off_vs); }
    float4* gbox() const { return reinterpret_cast<float4*>(ws + lay.off_gbox); }
    float4* sbox() const { return reinterpret_cast<float4*>(ws + lay.off_sbox); }
    template <class T> T* at(size_t off) const { return reinterpret_cast<T*>(ws + off); }
    // contact terms exist: gamma > 0 and some element has a radius at some step (with every radius 0 for good no pair can
    // touch, and the cell list would put a whole star into one cell)
    bool contact_on() const {
        return prm.gamma > 0.f && (prm.R_start[0] > 0.f || prm.R_start[1] > 0.f ||
                                   (prm.n_ramp > 0 && (prm.R_end[0] > 0.f || prm.R_end[1] > 0.f)));
    }
    int ngrav() const { return plan.sym_S ? (plan.chain ? 0 : plan.T) : plan.nsplit; }   // gravity slabs
    int ncontact() const {                                                // contact slabs
        if (!contact_on()) return 0;
        return contact_slabs(n);
    }
    int nslabs() const { return ngrav() + ncontact(); }                   // slabs nb_reduce_update_kernel sums
};

#define NB_CUDA(ctx, call)                                   \
    do {                                                     \
        cudaError_t e_ = (call);                             \
        if (e_ != cudaSuccess) { (ctx)->last_cuda = (int)e_; return NB_ECUDA; } \
    } while (0)

namespace {

// Every entry point that touches the device runs with the ctx's device current (nb.h: "dev" pointers belong to the
// device that was current at nb_create(), and so do the kernels' shared-memory opt-ins).
int device_guard(nb_ctx* c)
{
    int dev = -1;
    NB_CUDA(c, cudaGetDevice(&dev));
    return dev == c->device ? NB_OK : NB_ESTATE;
}

bool params_ok(const nb_params* p)
{
    auto fin = [](float x) { return std::isfinite(x); };
    if (!fin(p->G) || !fin(p->eps) || !fin(p->dt) || !fin(p->q) || !fin(p->gamma) || !fin(p->beta) ||
        !fin(p->v_dead))
        return false;
    if (p->G < 0.f || p->eps < 0.f || p->dt < 0.f) return false;
    if (!(p->q > 0.f && p->q <= 1.f)) return false;
    if (p->gamma < 0.f) return false;
    if (p->gamma > 0.f && !(p->beta > 0.f && p->beta <= 1.f)) return false;
    if (p->v_dead < 0.f) return false;
    if (p->n_ramp < 0) return false;
    if (p->lens_mode != 0 && p->lens_mode != 1) return false;
    for (int s = 0; s < 2; ++s)
        if (!fin(p->R_start[s]) || !fin(p->R_end[s]) || p->R_start[s] < 0.f || p->R_end[s] < 0.f) return false;
    return true;
}

// The instantiations of the symmetric kernel: <S, elements i per lane, threads, CTAs/SM, unroll>.
// 8 elements i per lane (254 registers, 8 warps per SM): a rotation step then carries 16 pair evaluations for its
// 6 SHFL + 3 LDS, and all 8 pairs' MUFU are in flight together (measured at N = 262,144: 4 i per lane / 16 warps
// 19.36 ms, 8 / 8 warps 18.41 ms, 8 / 12 warps at 168 registers 18.76 ms).
template <int S> struct SymShape;
template <> struct SymShape<256>  { static constexpr int NI = 4, NT = 64,  MINB = 8, UNR = 8; };   // small n: more, smaller CTAs win (16,384: 103 vs 113 us)
template <> struct SymShape<512>  { static constexpr int NI = 8, NT = 64,  MINB = 4, UNR = 16; };
template <> struct SymShape<1024> { static constexpr int NI = 8, NT = 128, MINB = 2, UNR = 16, kRounds = 1024 / (NT * NI); };   // (64 threads x 4 CTAs: 21.8 ms)
template <> struct SymShape<2048> { static constexpr int NI = 8, NT = 128, MINB = 2, UNR = 16, kRounds = 2048 / (NT * NI); };
template <> struct SymShape<4096> { static constexpr int NI = 8, NT = 128, MINB = 2, UNR = 16, kRounds = 4096 / (NT * NI); };

template <int S>
int launch_sym(nb_ctx* c, SymArgs& sa, int grid)
{
    using K = SymShape<S>;
    const int smem = kSymSmemPerElem * S;
    if (c->plan.chain) {                              // nb_kernels.cuh "Chain mode"
        auto kernel = nb_gravity_sym_chain_kernel<S, K::NI, K::NT, K::MINB, K::UNR>;   // shared-memory opt-in: configure_kernels()
        sa.acc64 = c->template at<double>(c->lay.off_acc64);
        sa.turn = c->template at<int>(c->lay.off_turn);
        constexpr int kRounds = S / (K::NT * K::NI);
        // turn counters and the ticket start at zero; the error word behind them is NOT cleared here: it is sticky from
        // nb_set_state() on, so a turn lost at step k of nb_step(100) is still there when the caller synchronises
        NB_CUDA(c, cudaMemsetAsync(sa.turn, 0, ((size_t)sa.T * (kRounds + 1) + 1) * sizeof(int), c->stream));
        kernel<<<grid, K::NT, smem, c->stream>>>(sa);
        c->chain_launched = true;
        return NB_OK;
    }
    auto kernel = nb_gravity_sym_kernel<S, K::NI, K::NT, K::MINB, K::UNR>;   // dynamic shared memory (112 KB at S = 4096)
    kernel<<<grid, K::NT, smem, c->stream>>>(sa);
    return NB_OK;
}

template <int S>
const char* sym_name(bool chain)
{
    using K = SymShape<S>;
    static char buf[2][72];
    std::snprintf(buf[chain], sizeof(buf[chain]), "nb_gravity_sym_%skernel<%d,%d,%d,%d,%d>", chain ? "chain_" : "", S, K::NI, K::NT,
                  K::MINB, K::UNR);
    return buf[chain];
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (kernel, DEVICE): every kernel that takes more than
// 48 KB of dynamic shared memory is opted in on the current device by nb_create(), once per ctx (a few host-side
// calls), not once per process -- a ctx created on a second GPU of the same process needs its own opt-in.
template <int S>
cudaError_t configure_sym()
{
    using K = SymShape<S>;
    const int smem = kSymSmemPerElem * S;
    cudaError_t e = cudaFuncSetAttribute(nb_gravity_sym_kernel<S, K::NI, K::NT, K::MINB, K::UNR>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    if (S >= 1024)
        e = cudaFuncSetAttribute(nb_gravity_sym_chain_kernel<S, K::NI, K::NT, K::MINB, K::UNR>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    return e;
}

cudaError_t configure_kernels()
{
    cudaError_t e;
    if ((e = configure_sym<256>()) != cudaSuccess) return e;
    if ((e = configure_sym<512>()) != cudaSuccess) return e;
    if ((e = configure_sym<1024>()) != cudaSuccess) return e;
    if ((e = configure_sym<2048>()) != cudaSuccess) return e;
    if ((e = configure_sym<4096>()) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(nb_pot_pair_kernel<4096, 8, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 4096)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(nb_pot_pair_kernel<8192, 8, 128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * 8192);
}

// Row a2: partial gravitational accelerations -> part[0..ngrav-1][n]
//   symmetric kernel: one CTA per pair of super-tiles, part[Y][e] = a_e due to super-tile Y
//   one-sided kernel: one CTA per (i-block, j-split), part[p][i] = a_i due to split p
int launch_gravity(nb_ctx* c)
{
    if (c->plan.sym_S) {
        SymArgs sa;
        sa.posm = c->posm; sa.part = c->part(); sa.acc64 = nullptr; sa.turn = nullptr; sa.n = (int)c->n; sa.T = c->plan.T;
        sa.G = c->prm.G; sa.eps = c->prm.eps;
        const long long T = c->plan.T;
        const int grid = (int)(T * (T + 1) / 2);
        int rc;
        if (c->plan.sym_S == 256)       rc = launch_sym<256>(c, sa, grid);
        else if (c->plan.sym_S == 512)  rc = launch_sym<512>(c, sa, grid);
        else if (c->plan.sym_S == 1024) rc = launch_sym<1024>(c, sa, grid);
        else if (c->plan.sym_S == 2048) rc = launch_sym<2048>(c, sa, grid);
        else                            rc = launch_sym<4096>(c, sa, grid);
        if (rc) return rc;
        c->launches++;
        NB_CUDA(c, cudaGetLastError());
        return NB_OK;
    }
    GravArgs ga;
    ga.posm = c->posm; ga.part = c->part();
    ga.n = (int)c->n; ga.nib = c->plan.nib; ga.nsplit = c->plan.nsplit; ga.njt = c->plan.njt;
    ga.G = c->prm.G; ga.eps = c->prm.eps;
    const int grid = c->plan.nib * c->plan.nsplit;
    if (c->plan.TJ == 256) nb_gravity_kernel<2, 256><<<grid, kThreads, 0, c->stream>>>(ga);
    else                   nb_gravity_kernel<2, 128><<<grid, kThreads, 0, c->stream>>>(ga);
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    return NB_OK;
}

// Launch `kernel` behind the previous kernel of the stream; with `pdl` as its programmatic dependent (the kernel
// starts launching before its predecessor has finished and waits for it in pdl_prologue()).
template <class... P, class... A>
cudaError_t launch_after(bool pdl, void (*kernel)(P...), int grid, int block, cudaStream_t st, A... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, P(args)...);
}

// Row a3: contact accelerations (Eqs. 5/6) of the pairs with r < R_i + R_j -> part[ngrav ...][n]
int launch_contact_on(nb_ctx* c, cudaStream_t st, double* epart = nullptr, unsigned long long* stats = nullptr)
{
    const int n = (int)c->n;
    ContactArgs ca;
    ca.ps = c->ps(); ca.vs = c->vs(); ca.perm = nullptr; ca.gbox = c->gbox(); ca.sbox = c->sbox();
    ca.out = c->part() + (size_t)c->ngrav() * c->n;
    ca.n = n;
    ca.gamma = c->prm.gamma; ca.gamma_beta = c->prm.gamma * c->prm.beta;
    ca.v_dead = c->prm.v_dead; ca.lens_mode = c->prm.lens_mode;
    if (c->n >= kCellMinN) {                                      // cell list (nb_cells.cuh)
        const Layout& L = c->lay;
        CellPassArgs a;
        a.posm = c->posm; a.vel = c->vel; a.dev = c->dev();
        a.part = c->at<CellPartial>(L.off_cpart); a.cs = c->at<CellState>(L.off_cstate);
        a.counters = c->at<int>(L.off_counters); a.bsum = c->at<int>(L.off_bsum);
        a.bucket = c->at<int>(L.off_bucket); a.slot = c->at<int>(L.off_slot); a.tmp = c->at<int>(L.off_tmp);
        a.perm = c->at<uint32_t>(L.off_perm); a.ps = c->ps(); a.vs = c->vs();
        a.out = ca.out; a.law = ca; a.epart = epart; a.stats = stats;
        a.n = n; a.n1 = c->n1;
        a.cap0 = (int)cell_cap(c->n1); a.cap1 = (int)cell_cap(c->n - c->n1); a.ncells = a.cap0 + a.cap1;
        a.lpe_log2 = c->n < kContactWideN ? 2 : 0;                  // lanes per element: 4 while the pass is latency-bound
        const long long eb = (n + kPassThreads - 1) / kPassThreads;
        long long cb;
        a.nparts = (int)(eb < kBoxBlocks ? eb : kBoxBlocks);
        const int sb = (a.ncells + kCellScanChunk - 1) / kCellScanChunk;
        const bool pdl = true;
        nb_cell_bbox_kernel<<<a.nparts, kPassThreads, 0, st>>>(a);
        NB_CUDA(c, launch_after(pdl, nb_cell_count_kernel, (int)eb, kPassThreads, st, a));
        NB_CUDA(c, launch_after(pdl, nb_cell_scan_kernel, sb, kPassThreads, st, a, 0));
        NB_CUDA(c, launch_after(pdl, nb_cell_scan_kernel, sb, kPassThreads, st, a, 3));
        NB_CUDA(c, launch_after(pdl, nb_cell_scatter_kernel, (int)eb, kPassThreads, st, a));
        NB_CUDA(c, launch_after(pdl, nb_cell_rank_kernel, (int)eb, kPassThreads, st, a));
        cb = (((long long)n << a.lpe_log2) + kCcThreads - 1) / kCcThreads;
        if (epart) {                                               // energy mode: U_rep partials instead of accelerations
            if (a.lpe_log2) NB_CUDA(c, launch_after(pdl, nb_contact_cell_kernel<2, true>, (int)cb, kCcThreads, st, a));
            else            NB_CUDA(c, launch_after(pdl, nb_contact_cell_kernel<0, true>, (int)cb, kCcThreads, st, a));
        } else if (stats) {                                        // counting mode (nb_contact_stats)
            if (a.lpe_log2) NB_CUDA(c, launch_after(pdl, nb_contact_cell_kernel<2, false, true>, (int)cb, kCcThreads, st, a));
            else            NB_CUDA(c, launch_after(pdl, nb_contact_cell_kernel<0, false, true>, (int)cb, kCcThreads, st, a));
        } else if (a.lpe_log2) {
            NB_CUDA(c, launch_after(pdl, nb_contact_cell_kernel<2>, (int)cb, kCcThreads, st, a));
        } else {
            NB_CUDA(c, launch_after(pdl, nb_contact_cell_kernel<0>, (int)cb, kCcThreads, st, a));
        }
        c->launches += 7;
        NB_CUDA(c, cudaGetLastError());
        return NB_OK;
    }
    // small n: groups of 32 in index order, every group a candidate of every other
    const int ngroups = (n + kGroup - 1) / kGroup;
    const int nsuper = (ngroups + kSuper - 1) / kSuper;
    nb_gather_kernel<<<nsuper, kGroup * kSuper, 0, st>>>(c->posm, c->vel, nullptr, n, c->dev(), c->ps(), c->vs(),
                                                               c->gbox(), c->sbox());
    c->launches++;
    ca.ngroups = ngroups; ca.nsuper = nsuper;
    const int nchunks = c->ncontact();
    const long long warps = (long long)ngroups * nchunks;
    ca.nchunks = nchunks;
    const int cg = (ngroups + nchunks - 1) / nchunks;
    nb_contact_chunk_kernel<<<(int)((warps * 32 + kThreads - 1) / kThreads), kThreads, 0, st>>>(ca, cg, nchunks);
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    return NB_OK;
}

int launch_contact(nb_ctx* c) { return launch_contact_on(c, c->stream); }

// Rows a2 + a3: every slab nb_reduce_update_kernel sums for a(x).  The two are independent (both
// read the state, each writes its own slabs), so the contact pass -- seven short launches that
// cannot fill the machine -- runs on the library's side stream: fork after whatever the ctx stream
// holds, join before the update kernel.  The gravity kernel is launched FIRST and the side stream has
// the same (default) priority, so the block scheduler places the contact CTAs where the gravity kernel
// leaves room: beside the one-sided kernel, and in the ragged last wave of the symmetric kernel, whose
// CTAs fill the register file (measured whole steps, contact first on a high-priority stream -> this
// order: 16,384 elements 156 -> 135 us, 65,536 1.322 -> 1.280 ms, 262,144 18.81 -> 18.64 ms; a contact
// CTA that takes a slot from a retiring gravity CTA mid-kernel costs more than it would in the tail).
int launch_force(nb_ctx* c)
{
    if (!c->contact_on()) return launch_gravity(c);
    NB_CUDA(c, cudaEventRecord(c->ev_fork, c->stream));
    int rc = launch_gravity(c);
    if (rc) return rc;
    NB_CUDA(c, cudaStreamWaitEvent(c->side, c->ev_fork, 0));
    rc = launch_contact_on(c, c->side);
    if (rc) return rc;
    NB_CUDA(c, cudaEventRecord(c->ev_join, c->side));
    NB_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_join, 0));
    return NB_OK;
}

// Rows a4+a6+a5: reduce `nsrc` slabs of `src`, optionally store a, kick, drift, advance.
int launch_update(nb_ctx* c, const float4* src, int nsrc, float4* acc_out, float kick_h, float drift_dt,
                  int advance, float vscale = 1.f)
{
    UpdateArgs u;
    u.acc64 = (src == c->part() && c->plan.sym_S && c->plan.chain) ? c->at<double>(c->lay.off_acc64) : nullptr;
    u.src = src; u.acc_out = acc_out; u.posm = c->posm; u.vel = c->vel; u.dev = c->dev();
    u.n = (int)c->n; u.nsrc = nsrc; u.kick_h = kick_h; u.drift_dt = drift_dt; u.advance = advance; u.vscale = vscale;
    const int grid = (int)((c->n + 255) / 256);
    nb_reduce_update_kernel<<<grid, 256, 0, c->stream>>>(u);
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    return NB_OK;
}

// n < kCellMinN: rows a2-a6 for `nforce` force evaluations in ONE cooperative launch (nb_fused.cuh).
bool fused_path(const nb_ctx* c) { return c->n < kCellMinN && !c->plan.sym_S && c->fused_blocks > 0; }

int launch_fused(nb_ctx* c, int nforce, int open, int close_mode, float4* acc_out, bool relax = false, float vscale = 1.f)
{
    FusedArgs f;
    std::memset(&f, 0, sizeof(f));
    const int n = (int)c->n;
    f.posm = c->posm; f.vel = c->vel; f.posm2 = c->ps(); f.vel2 = c->vs();      // the contact pass's sorted copies are free here
    f.acc = c->acc(); f.acc_out = acc_out; f.dev = c->dev();
    f.law.n = n;
    f.law.gamma = c->prm.gamma; f.law.gamma_beta = c->prm.gamma * c->prm.beta;
    f.law.v_dead = c->prm.v_dead; f.law.lens_mode = c->prm.lens_mode;
    f.n = n; f.n1 = c->n1; f.G = c->prm.G; f.eps = c->prm.eps; f.dt = c->prm.dt;
    f.nforce = nforce; f.open = open; f.close_mode = close_mode; f.relax = relax ? 1 : 0; f.vscale = vscale;
    f.logP = c->fused_logP; f.npad = (n + kFusedGroup - 1) & ~(kFusedGroup - 1);
    void* args[] = {&f};
    NB_CUDA(c, cudaLaunchCooperativeKernel((const void*)nb_fused_step_kernel, dim3((unsigned)c->fused_blocks), dim3(kFusedThreads),
                                           args, fused_smem_bytes(n), c->stream));
    c->launches++;
    return NB_OK;
}

// Shape of the fused kernel for the bound state: the smallest power of two P (packed pairs of elements i per CTA)
// whose ceil(n / 2P) CTAs are all co-resident (the kernel synchronises grid-wide); fused_blocks = 0 if none is.
void plan_fused(nb_ctx* c)
{
    c->fused_blocks = 0;
    if (!c->fused_ok || c->n >= kCellMinN) return;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, nb_fused_step_kernel, kFusedThreads,
                                                      fused_smem_bytes(c->n)) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return;
    }
    const int64_t cap = (int64_t)per_sm * c->num_sms;
    for (int lp = 0; lp <= kFusedMaxLogP; ++lp) {
        const int64_t blocks = (c->n + (2LL << lp) - 1) / (2LL << lp);
        if (blocks <= cap) { c->fused_logP = lp; c->fused_blocks = (int)blocks; return; }
    }
}

// Chain mode: a turn that never came (it cannot, by the ticket order -- this is the safety net that keeps a bug from
// hanging the GPU) raises a flag on the device; the synchronising entry points report it.
int chain_flag_check(nb_ctx* c)
{
    if (!c->have_state || !c->plan.sym_S || !c->plan.chain || !c->chain_launched) return NB_OK;
    const int S = c->plan.sym_S;
    const int rounds = S == 1024 ? SymShape<1024>::kRounds : (S == 2048 ? SymShape<2048>::kRounds : SymShape<4096>::kRounds);
    int flag = 0;
    NB_CUDA(c, cudaMemcpyAsync(&flag, c->at<int>(c->lay.off_turn) + (size_t)c->plan.T * (rounds + 1) + 1, sizeof(int),
                               cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    if (flag) {                                          // sums added out of turn: a(x) and everything stepped with it is void
        c->have_acc = false;
        c->last_cuda = (int)cudaErrorLaunchTimeout;
        return NB_ECUDA;
    }
    return NB_OK;
}

int ensure_acc(nb_ctx* c)
{
    if (c->have_acc) return NB_OK;
    if (fused_path(c)) {
        const int rc = launch_fused(c, 1, 0, 1, nullptr);
        if (rc) return rc;
        c->have_acc = true; c->acc_uploaded = false;
        return NB_OK;
    }
    int rc = launch_force(c);
    if (rc) return rc;
    rc = launch_update(c, c->part(), c->nslabs(), c->acc(), 0.f, 0.f, 0);
    if (rc) return rc;
    c->have_acc = true; c->acc_uploaded = false;
    return NB_OK;
}

}  // namespace

extern "C" {

const char* nb_strerror(int status)
{
    switch (status) {
        case NB_OK: return "ok";
        case NB_EINVAL: return "invalid argument";
        case NB_ESTATE: return "invalid state or call order (no state bound, or star[] is not 0...0 1...1)";
        case NB_ECUDA: return "CUDA error (see nb_last_cuda_error)";
        case NB_ENOMEM: return "workspace too small or host allocation failed";
        case NB_EARCH: return "device is not sm_100 (B200)";
        case NB_ESIZE: return "n exceeds nb_gravity_accel_static_max_n(): the entry point without a workspace has a fixed scratch array; use the ctx API";
        default: return "unknown status";
    }
}

int nb_last_cuda_error(nb_ctx* ctx) { return ctx ? ctx->last_cuda : 0; }

size_t nb_workspace_bytes(int64_t n_max)
{
    if (n_max < 1 || n_max > kMaxN) return 0;
    return make_layout(n_max).total;
}

int nb_create(nb_ctx** out, int64_t n_max, const nb_params* p, void* cuda_stream)
{
    if (!out) return NB_EINVAL;
    *out = nullptr;
    if (!p || n_max < 1 || n_max > kMaxN || !params_ok(p)) return NB_EINVAL;
    int dev = 0, major = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return NB_ECUDA;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return NB_ECUDA;
    if (major != 10) return NB_EARCH;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return NB_ECUDA;
    nb_ctx* c = new (std::nothrow) nb_ctx();
    if (!c) return NB_ENOMEM;
    c->prm = *p;
    c->n_max = n_max;
    c->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    c->num_sms = sms > 0 ? sms : kNumSMsFallback;
    c->device = dev;
    c->lay = make_layout(n_max);
    {
        const cudaError_t e = configure_kernels();
        if (e != cudaSuccess) { cudaGetLastError(); delete c; return NB_ECUDA; }
    }
    // default priority, like the gravity kernel launched before it: see launch_force()
    if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        nb_destroy(c);
        return NB_ECUDA;
    }
    {   // the fused small-n kernel: a cooperative launch with up to ~200 KB of dynamic shared memory
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        c->fused_ok = coop && cudaFuncSetAttribute(nb_fused_step_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                   (int)fused_smem_bytes(kCellMinN - 1)) == cudaSuccess;
        if (!c->fused_ok) cudaGetLastError();
    }
    *out = c;
    return NB_OK;
}

void nb_destroy(nb_ctx* ctx)
{
    if (!ctx) return;
    if (ctx->side) { cudaStreamSynchronize(ctx->side); cudaStreamDestroy(ctx->side); }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    delete ctx;
}

int nb_set_state(nb_ctx* c, int64_t n, float* posm, float* vel, const int32_t* star, void* workspace,
                 size_t workspace_bytes)
{
    if (!c || !posm || !vel || !star || !workspace) return NB_EINVAL;
    if (n < 1 || n > c->n_max) return NB_EINVAL;
    if (((uintptr_t)posm & 15) || ((uintptr_t)vel & 15) || ((uintptr_t)star & 3) ||
        ((uintptr_t)workspace & (kAlign - 1)))
        return NB_EINVAL;
    if (workspace_bytes < c->lay.total) return NB_ENOMEM;
    if (int rc_ = device_guard(c)) return rc_;
    c->have_state = false;
    c->have_acc = false;
    c->acc_uploaded = false;
    c->chain_launched = false;
    c->ws = static_cast<char*>(workspace);

    DevState h;
    std::memset(&h, 0, sizeof(h));
    for (int s = 0; s < 2; ++s) {
        h.R_start[s] = (double)c->prm.R_start[s];
        h.R_end[s] = (double)c->prm.R_end[s];
        h.R[s] = c->prm.R_start[s];
    }
    h.n_ramp = c->prm.n_ramp;
    NB_CUDA(c, cudaMemcpyAsync(c->dev(), &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
    nb_validate_star_kernel<<<c->num_sms, 256, 0, c->stream>>>(star, (int)n, c->dev());
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    NB_CUDA(c, cudaMemcpyAsync(&h, c->dev(), sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    if (h.bad) return NB_ESTATE;
    // chain mode's turn counters, ticket and ERROR WORD: all zero from here on; the launches clear the counters and the
    // ticket again, nothing but this call clears the error word (its position depends on n only)
    if (c->n_max >= kChainMinN)
        NB_CUDA(c, cudaMemsetAsync(c->at<int>(c->lay.off_turn), 0, ((size_t)(c->n_max / 1024 + 1) * 5 + 2) * sizeof(int), c->stream));

    c->n = n;
    c->n1 = h.n1;
    c->posm = reinterpret_cast<float4*>(posm);
    c->vel = reinterpret_cast<float4*>(vel);
    c->plan = make_plan(n, c->num_sms, c->path);
    if ((int64_t)c->nslabs() * n > partial_elems_bound(c->n_max)) return NB_ENOMEM;
    plan_fused(c);
    c->have_state = true;
    return NB_OK;
}

int nb_compute_accel(nb_ctx* c, float* acc)
{
    if (!c || !acc || ((uintptr_t)acc & 15)) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    if (fused_path(c)) {
        const int rc = launch_fused(c, 1, 0, 1, reinterpret_cast<float4*>(acc) != c->acc() ? reinterpret_cast<float4*>(acc) : nullptr);
        if (rc) return rc;
        c->have_acc = true; c->acc_uploaded = false;
        return NB_OK;
    }
    int rc = launch_force(c);
    if (rc) return rc;
    rc = launch_update(c, c->part(), c->nslabs(), reinterpret_cast<float4*>(acc), 0.f, 0.f, 0);
    if (rc) return rc;
    if (reinterpret_cast<float4*>(acc) != c->acc()) {
        NB_CUDA(c, cudaMemcpyAsync(c->acc(), acc, (size_t)c->n * sizeof(float4), cudaMemcpyDeviceToDevice,
                                   c->stream));
    }
    c->have_acc = true; c->acc_uploaded = false;
    return NB_OK;
}

int nb_step(nb_ctx* c, int nsteps)
{
    if (!c || nsteps < 0) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    if (nsteps == 0) return NB_OK;
    const float dt = c->prm.dt;
    int rc = ensure_acc(c);                                    // a(x_n) with v_n (A7)
    if (rc) return rc;
    if (fused_path(c)) return launch_fused(c, nsteps, 1, 0, nullptr);   // all nsteps in one launch
    // v_{n+1/2} = v_n + dt/2 a_n ; x_{n+1} = x_n + dt v_{n+1/2} ; n += 1, R(n)
    rc = launch_update(c, c->acc(), 1, nullptr, 0.5f * dt, dt, 1);
    if (rc) return rc;
    for (int s = 1; s <= nsteps; ++s) {
        rc = launch_force(c);                                  // a(x_{n+s}) with v_{n+s-1/2}
        if (rc) return rc;
        if (s < nsteps)   // two half kicks merged: v += dt a ; x += dt v ; advance
            rc = launch_update(c, c->part(), c->nslabs(), nullptr, dt, dt, 1);
        else              // closing half kick; cache a(x_{n+nsteps})
            rc = launch_update(c, c->part(), c->nslabs(), c->acc(), 0.5f * dt, 0.f, 0);
        if (rc) return rc;
    }
    c->have_acc = true; c->acc_uploaded = false;
    return NB_OK;
}

int nb_relax(nb_ctx* c, int nsteps, float kappa)
{
    if (!c || nsteps < 0 || !(kappa >= 0.f) || !std::isfinite(kappa)) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    if (nsteps == 0) return NB_OK;
    const float dt = c->prm.dt;
    float f = 1.f - kappa * dt;                               // rounded as written: one multiply, one subtract
    if (!(f > 0.f)) f = 0.f;
    int rc = ensure_acc(c);
    if (rc) return rc;
    if (fused_path(c)) return launch_fused(c, nsteps, 1, 0, nullptr, true, f);   // all nsteps in one launch
    for (int s = 0; s < nsteps; ++s) {
        rc = launch_update(c, c->acc(), 1, nullptr, 0.5f * dt, dt, 1);          // half kick, drift, n += 1
        if (rc) return rc;
        rc = launch_force(c);
        if (rc) return rc;
        rc = launch_update(c, c->part(), c->nslabs(), c->acc(), 0.5f * dt, 0.f, 0, f);   // half kick, then v <- f v
        if (rc) return rc;
    }
    c->have_acc = true; c->acc_uploaded = false;
    return NB_OK;
}

// f3 on the device: pass 1 (star moments), geometry (centres, L1 plane, Eq. 3 lobes), pass 2 (decisions), record.
// Four launches on the ctx stream, nothing synchronises.
static int launch_transfer(nb_ctx* c, double k_lobe, double* series, long long rows)
{
    const int n = (int)c->n;
    double* red = c->red();
    XferGeom* g = c->at<XferGeom>(c->lay.off_xfer);
    nb_star_moments_kernel<<<kMomentBlocks, 256, 0, c->stream>>>(c->posm, c->vel, n, c->n1, red);
    nb_transfer_geometry_kernel<<<1, 32, 0, c->stream>>>(red, kMomentBlocks, k_lobe, c->dev(), series, rows, g);
    XferArgs xa;
    xa.posm = c->posm; xa.vel = c->vel; xa.g = g; xa.out = red; xa.n = n; xa.n1 = c->n1;
    nb_transfer_kernel<<<kMomentBlocks, 256, 0, c->stream>>>(xa);
    nb_transfer_finish_kernel<<<1, 32, 0, c->stream>>>(red, kMomentBlocks, g);
    c->launches += 4;
    NB_CUDA(c, cudaGetLastError());
    return NB_OK;
}

int nb_transfer_diagnostics(nb_ctx* c, double k_lobe, double* out)
{
    if (!c || !out || !(k_lobe > 0.0) || !std::isfinite(k_lobe)) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    double* row = reinterpret_cast<double*>(c->ws + c->lay.off_xfer + align_up(sizeof(XferGeom)));
    if (int rc = launch_transfer(c, k_lobe, row, -1)) return rc;
    NB_CUDA(c, cudaMemcpyAsync(out, row, 32 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    return NB_OK;
}

int nb_transfer_record(nb_ctx* c, double k_lobe, double* dev_series, int64_t rows)
{
    if (!c || !dev_series || rows < 1 || ((uintptr_t)dev_series & 7) || !(k_lobe > 0.0) || !std::isfinite(k_lobe)) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    return launch_transfer(c, k_lobe, dev_series, (long long)rows);
}

int nb_splat(nb_ctx* c, const float* centre, float half_width, int axis_u, int axis_v, int W, int H,
             uint32_t* image)
{
    if (!c || !centre || !image || !(half_width > 0.f) || !std::isfinite(half_width)) return NB_EINVAL;
    if (axis_u < 0 || axis_u > 2 || axis_v < 0 || axis_v > 2 || axis_u == axis_v) return NB_EINVAL;
    if (W < 1 || H < 1 || W > 16384 || H > 16384 || ((uintptr_t)image & 3)) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    const float scale = (float)W / (2.0f * half_width);        // pixels per unit length, fp32
    NB_CUDA(c, cudaMemsetAsync(image, 0, (size_t)2 * W * H * sizeof(uint32_t), c->stream));
    nb_splat_kernel<<<(int)((c->n + 255) / 256), 256, 0, c->stream>>>(c->posm, (int)c->n, c->n1, centre[axis_u],
                                                                     centre[axis_v], scale, axis_u, axis_v, W, H, image);
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    return NB_OK;
}

int nb_get_step(nb_ctx* c, int64_t* step, float* R)
{
    if (!c) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    DevState h;
    NB_CUDA(c, cudaMemcpyAsync(&h, c->dev(), sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    if (const int rc = chain_flag_check(c)) return rc;
    if (step) *step = h.step;
    if (R) { R[0] = h.R[0]; R[1] = h.R[1]; }
    return NB_OK;
}

int nb_set_step(nb_ctx* c, int64_t step)
{
    if (!c || step < 0) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    nb_set_step_kernel<<<1, 1, 0, c->stream>>>(c->dev(), (long long)step);
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    // A cached a(x) holds contact terms at the radii of the step it was evaluated at.  It stays only when it cannot be
    // stale: the radii do not move with the step count, or it was uploaded with the checkpoint this call completes.
    const bool radii_move = c->contact_on() && c->prm.n_ramp > 0 &&
                            (c->prm.R_start[0] != c->prm.R_end[0] || c->prm.R_start[1] != c->prm.R_end[1]);
    if (radii_move && !c->acc_uploaded) c->have_acc = false;
    return NB_OK;
}

int nb_energy(nb_ctx* c, double* out)
{
    if (!c || !out) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    int rc = ensure_acc(c);
    if (rc) return rc;
    rc = chain_flag_check(c);
    if (rc) return rc;
    const int n = (int)c->n;
    double* red_m = c->red();
    double* red_p = red_m + (size_t)kMomentBlocks * kMomentCols;
    nb_moments_kernel<<<kMomentBlocks, 256, 0, c->stream>>>(c->posm, c->vel, c->acc(), n, red_m);
    c->launches++;
    NB_CUDA(c, cudaGetLastError());
    size_t npot = 0, nrep = 0;                       // fp64 partials: U_grav (x 2 with U_rep interleaved for small n), U_rep
    double *dpot = nullptr, *drep = nullptr;
    const bool big = c->n >= kCellMinN;
    if (big) {                                       // packed pair-of-super-tiles kernel + the cell list in energy mode
        // U_rep first: the cell list in energy mode, which also leaves the elements in cell order (ps, vs) -- the
        // order in which most pairs of super-tiles are far apart (nb_pot_pair_kernel)
        if (c->contact_on()) {
            drep = c->at<double>(c->lay.off_erep);
            nrep = (size_t)((((long long)n << (c->n < kContactWideN ? 2 : 0)) + kCcThreads - 1) / kCcThreads);
            rc = launch_contact_on(c, c->stream, drep);
            if (rc) return rc;
        }
        PotPairArgs pa;
        pa.px = c->contact_on() ? c->ps() : c->posm;
        pa.pm = c->contact_on() ? c->vs() : c->posm;
        pa.out = dpot = c->at<double>(c->lay.off_epot);
        pa.n = n; pa.G = c->prm.G; pa.eps = c->prm.eps;
        const int S = pot_tile(c->n);
        pa.T = (int)((c->n + S - 1) / S);
        npot = (size_t)pot_pairs(c->n);
        float4* tbox = c->at<float4>(c->lay.off_tbox);
        pa.box = tbox;
        nb_tile_bbox_kernel<<<pa.T, 256, 0, c->stream>>>(pa.px, n, S, tbox);
        c->launches++;
        if (S == 1024)      nb_pot_pair_kernel<1024, 8, 128><<<(unsigned)npot, 128, 16 * 1024, c->stream>>>(pa);
        else if (S == 4096) nb_pot_pair_kernel<4096, 8, 128><<<(unsigned)npot, 128, 16 * 4096, c->stream>>>(pa);   // > 48 KB: configure_kernels()
        else                nb_pot_pair_kernel<8192, 8, 128><<<(unsigned)npot, 128, 16 * 8192, c->stream>>>(pa);
        c->launches++;
        NB_CUDA(c, cudaGetLastError());
    } else {
        const int pot_blocks = (n + kThreads - 1) / kThreads;
        PotArgs pa;
        pa.posm = c->posm; pa.dev = c->dev(); pa.out = dpot = red_p; pa.n = n; pa.n1 = c->n1;
        pa.G = c->prm.G; pa.eps = c->prm.eps; pa.gamma = c->prm.gamma;
        nb_potential_kernel<<<pot_blocks, kThreads, 0, c->stream>>>(pa);
        c->launches++;
        NB_CUDA(c, cudaGetLastError());
        npot = (size_t)pot_blocks * 2;
    }

    const size_t nm = (size_t)kMomentBlocks * kMomentCols;
    double* h = new (std::nothrow) double[nm + npot + nrep];
    if (!h) return NB_ENOMEM;
    DevState hs;
    cudaError_t e = cudaMemcpyAsync(h, red_m, nm * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h + nm, dpot, npot * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess && nrep) e = cudaMemcpyAsync(h + nm + npot, drep, nrep * sizeof(double), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&hs, c->dev(), sizeof(hs), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { delete[] h; c->last_cuda = (int)e; return NB_ECUDA; }
    double m[kMomentCols] = {0};
    for (int b = 0; b < kMomentBlocks; ++b)
        for (int k = 0; k < kMomentCols; ++k) m[k] += h[(size_t)b * kMomentCols + k];
    double ug2 = 0.0, ur2 = 0.0;
    const double* hp = h + nm;
    if (big) {
        for (size_t b = 0; b < npot; ++b) ug2 += hp[b];
        for (size_t b = 0; b < nrep; ++b) ur2 += hp[npot + b];
    } else {
        for (size_t b = 0; b < npot / 2; ++b) { ug2 += hp[2 * b]; ur2 += hp[2 * b + 1]; }
    }
    delete[] h;
    out[0] = m[0];
    out[1] = -ug2;
    out[2] = ur2;
    out[3] = out[0] + out[1] + out[2];
    for (int k = 0; k < 6; ++k) out[4 + k] = m[1 + k];
    out[10] = std::sqrt(m[7] * m[7] + m[8] * m[8] + m[9] * m[9]);
    out[11] = (double)hs.step;
    return NB_OK;
}

int nb_upload_state(nb_ctx* c, const float* host_posm, const float* host_vel, const float* host_acc)
{
    if (!c) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    const size_t bytes = (size_t)c->n * sizeof(float4);
    if (host_posm) NB_CUDA(c, cudaMemcpyAsync(c->posm, host_posm, bytes, cudaMemcpyHostToDevice, c->stream));
    if (host_vel) NB_CUDA(c, cudaMemcpyAsync(c->vel, host_vel, bytes, cudaMemcpyHostToDevice, c->stream));
    if (host_acc) NB_CUDA(c, cudaMemcpyAsync(c->acc(), host_acc, bytes, cudaMemcpyHostToDevice, c->stream));
    c->have_acc = host_acc != nullptr;
    c->acc_uploaded = c->have_acc;
    return NB_OK;
}

int nb_download_state(nb_ctx* c, float* host_posm, float* host_vel, float* host_acc)
{
    if (!c) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    const size_t bytes = (size_t)c->n * sizeof(float4);
    if (host_acc) {
        const int rc = ensure_acc(c);
        if (rc) return rc;
        NB_CUDA(c, cudaMemcpyAsync(host_acc, c->acc(), bytes, cudaMemcpyDeviceToHost, c->stream));
    }
    if (host_posm) NB_CUDA(c, cudaMemcpyAsync(host_posm, c->posm, bytes, cudaMemcpyDeviceToHost, c->stream));
    if (host_vel) NB_CUDA(c, cudaMemcpyAsync(host_vel, c->vel, bytes, cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    return chain_flag_check(c);
}

int nb_get_launch_info(nb_ctx* c, int32_t* out4)
{
    if (!c || !out4) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    if (fused_path(c)) {                  // one cooperative launch: elements i per CTA, j segments per CTA, CTAs
        out4[0] = 2 << c->fused_logP;
        out4[1] = kFusedThreads >> c->fused_logP;
        out4[2] = out4[3] = c->fused_blocks;
        return NB_OK;
    }
    if (c->plan.sym_S) {
        out4[0] = c->plan.sym_S;
        out4[1] = c->plan.T;
        out4[2] = (int)((long long)c->plan.T * (c->plan.T + 1) / 2);
    } else {
        out4[0] = kThreads * c->plan.I;
        out4[1] = c->plan.nsplit;
        out4[2] = c->plan.nib * c->plan.nsplit;
    }
    out4[3] = (int)((c->n + 255) / 256);
    return NB_OK;
}

int nb_set_force_path(nb_ctx* c, int path)
{
    if (!c || path < kPathAuto || path > kPathSymmetric) return NB_EINVAL;
    if (c->have_state) {
        const Plan p = make_plan(c->n, c->num_sms, path);
        const int64_t ngrav = p.sym_S ? (p.chain ? 0 : p.T) : p.nsplit;
        if ((ngrav + c->ncontact()) * c->n > partial_elems_bound(c->n_max)) return NB_ENOMEM;
        c->plan = p;
    }
    c->path = path;
    return NB_OK;
}

const char* nb_force_kernel_name(nb_ctx* c)
{
    if (!c || !c->have_state) return "";
    if (fused_path(c)) return "nb_fused_step_kernel";          // rows a2-a6 in one launch (its loop is the one-sided one)
    if (c->plan.sym_S == 256) return sym_name<256>(c->plan.chain);
    if (c->plan.sym_S == 512) return sym_name<512>(c->plan.chain);
    if (c->plan.sym_S == 1024) return sym_name<1024>(c->plan.chain);
    if (c->plan.sym_S == 2048) return sym_name<2048>(c->plan.chain);
    if (c->plan.sym_S) return sym_name<4096>(c->plan.chain);
    return c->plan.TJ == 256 ? "nb_gravity_kernel<2,256>" : "nb_gravity_kernel<2,128>";
}

int64_t nb_launch_count(nb_ctx* c) { return c ? c->launches : 0; }

namespace {
int time_launches(nb_ctx* c, int reps, float* ms_avg, int (*launch)(nb_ctx*))
{
    if (!c || !ms_avg || reps < 1) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    cudaEvent_t e0, e1;
    NB_CUDA(c, cudaEventCreate(&e0));
    NB_CUDA(c, cudaEventCreate(&e1));
    int rc = launch(c);                                        // warm-up, untimed
    if (rc == NB_OK) {
        cudaEventRecord(e0, c->stream);
        for (int r = 0; r < reps && rc == NB_OK; ++r) rc = launch(c);
        cudaEventRecord(e1, c->stream);
    }
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc) return rc;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return NB_ECUDA; }
    *ms_avg = ms / (float)reps;
    return NB_OK;
}
}  // namespace

int nb_contact_stats(nb_ctx* c, int64_t* out2)
{
    if (!c || !out2) return NB_EINVAL;
    if (!c->have_state) return NB_ESTATE;
    if (int rc_ = device_guard(c)) return rc_;
    out2[0] = out2[1] = 0;
    if (!c->contact_on()) return NB_OK;
    if (c->n < kCellMinN) {                                    // no cell list: every ordered pair is pre-tested
        out2[0] = c->n * (c->n - 1);
        out2[1] = -1;
        return NB_OK;
    }
    unsigned long long* d = reinterpret_cast<unsigned long long*>(c->at<double>(c->lay.off_erep));
    NB_CUDA(c, cudaMemsetAsync(d, 0, 2 * sizeof(unsigned long long), c->stream));
    int rc = launch_contact_on(c, c->stream, nullptr, d);
    if (rc) return rc;
    unsigned long long h[2] = {0, 0};
    NB_CUDA(c, cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    NB_CUDA(c, cudaStreamSynchronize(c->stream));
    out2[0] = (int64_t)h[0]; out2[1] = (int64_t)h[1];
    return NB_OK;
}

int nb_time_force_kernel(nb_ctx* c, int reps, float* ms_avg)
{
    return time_launches(c, reps, ms_avg, launch_gravity);
}

int nb_time_contact_pass(nb_ctx* c, int reps, float* ms_avg)
{
    if (c && !c->contact_on()) { if (ms_avg) *ms_avg = 0.f; return c->have_state ? NB_OK : NB_ESTATE; }
    return time_launches(c, reps, ms_avg, launch_contact);
}

double nb_roche_lobe_radius(double mass_ratio, double k)
{
    if (!(mass_ratio > 0.0) || !std::isfinite(mass_ratio) || !(k > 0.0)) return NAN;
    const double c = std::cbrt(mass_ratio);
    return 0.49 * c * c / (k * c * c + std::log1p(c));           // Eq. 3
}

double nb_l1_distance(double q)
{
    if (!(q > 0.0) || !(q <= 1.0)) return NAN;
    // Newton iteration on the co-rotating force balance along the line of centres
    // (separation 1, G(m1+m2) = 1): s = distance from the primary m1.
    const double mu2 = q / (1.0 + q), mu1 = 1.0 - mu2;
    double s = 1.0 - std::cbrt(mu2 / 3.0);                        // Hill-radius start
    for (int it = 0; it < 100; ++it) {
        const double t = 1.0 - s;
        const double f = -mu1 / (s * s) + mu2 / (t * t) + (s - mu2);
        const double df = 2.0 * mu1 / (s * s * s) + 2.0 * mu2 / (t * t * t) + 1.0;
        const double sn = s - f / df;
        if (!(sn > 0.0 && sn < 1.0)) { s = 0.5 * (s + (sn <= 0.0 ? 0.0 : 1.0)); continue; }
        if (std::fabs(sn - s) < 1e-15) { s = sn; break; }
        s = sn;
    }
    return s;
}


// ---------------------------------------------------------------------------------------------------------
// nb_gravity_accel_static(): row a2 (Eq. 4, summed over all pairs) for callers
// that have no way to get device memory for a workspace -- see include/nb.h for who they are.  The
// one-sided gravity kernel needs scratch: a CTA owns an (i-block, j-split) and writes the partial
// acceleration of its elements i due to its split of the elements j into slab `split` of n float4;
// nb_reduce_update_kernel then adds the slabs of an element in split order.  Everywhere else those slabs sit
// in the caller's workspace; here they sit in the array below, which is part of the library image: the
// driver places it on every device that loads this module and keeps it there until the process ends.
namespace {

constexpr int64_t kStaticMaxN = 16384;                       // largest n the entry point takes
constexpr int64_t kStaticSlots = 8 * kStaticMaxN;            // float4 partial sums: 2 MiB; n * splits <= this
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) float4 nb_static_scratch[kStaticSlots];

// In host code `nb_static_scratch` is only a handle for the runtime's symbol calls -- it is NOT the array's
// device address, and a kernel handed `nb_static_scratch` from the host side would write somewhere else or
// fault.  The address a kernel can use comes from cudaGetSymbolAddress(), differs from device to device,
// and is looked up once per device (with that device current) and kept here.
struct StaticDevice {
    float4* scratch = nullptr;
    int num_sms = 0;
    bool ready = false;
};
StaticDevice g_static_device[kStaticMaxDevices];
std::mutex g_static_mutex;

// Per-device set-up of the first call on the current device.  Allocates nothing.
int static_device(const StaticDevice** out, cudaError_t* err)
{
    int dev = -1;
    if ((*err = cudaGetDevice(&dev)) != cudaSuccess) return NB_ECUDA;
    if (dev < 0 || dev >= kStaticMaxDevices) return NB_EINVAL;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_device[dev];
    if (!d.ready) {
        int major = 0, sms = 0;
        if ((*err = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess) return NB_ECUDA;
        if (major != 10) return NB_EARCH;
        if ((*err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return NB_ECUDA;
        float4* ptr = nullptr;
        if ((*err = cudaGetSymbolAddress((void**)&ptr, nb_static_scratch)) != cudaSuccess) return NB_ECUDA;
        if (!ptr) { *err = cudaErrorInvalidSymbol; return NB_ECUDA; }
        d.scratch = ptr;
        d.num_sms = sms > 0 ? sms : kNumSMsFallback;
        d.ready = true;
    }
    *out = &d;
    return NB_OK;
}

}  // namespace

int64_t nb_gravity_accel_static_max_n(void) { return kStaticMaxN; }

int nb_gravity_accel_static(int64_t n, const float* posm, float G, float eps, float* acc, void* cuda_stream, int* cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    if (!posm || !acc || n < 1) return NB_EINVAL;
    if (n > kStaticMaxN) return NB_ESIZE;                    // before anything touches the device
    if ((reinterpret_cast<uintptr_t>(posm) | reinterpret_cast<uintptr_t>(acc)) & 15u) return NB_EINVAL;
    if (!std::isfinite(G) || !std::isfinite(eps) || G < 0.f || eps < 0.f) return NB_EINVAL;
    cudaError_t err = cudaSuccess;
    auto fail = [&](int rc) { if (cuda_error) *cuda_error = (int)err; return rc; };
    const StaticDevice* d = nullptr;
    if (int rc = static_device(&d, &err)) return fail(rc);
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);

    // the one-sided plan of the ctx API, with its j splits cut to what the fixed array holds
    Plan p = make_plan(n, d->num_sms, kPathOneSided);
    const int64_t room = kStaticSlots / n;                   // >= 8
    if (p.nsplit > room) p.nsplit = (int)room;
    if (p.nsplit > p.njt) p.nsplit = p.njt;                  // every split holds at least one tile
    GravArgs ga;
    ga.posm = reinterpret_cast<const float4*>(posm); ga.part = d->scratch;
    ga.n = (int)n; ga.nib = p.nib; ga.nsplit = p.nsplit; ga.njt = p.njt;
    ga.G = G; ga.eps = eps;
    const int grid = p.nib * p.nsplit;
    // every slot [split][i], i < n, split < nsplit, is written here before the reduction reads it: whatever an
    // earlier call left in the array is never seen
    if (p.TJ == 256) nb_gravity_kernel<2, 256><<<grid, kThreads, 0, st>>>(ga);
    else             nb_gravity_kernel<2, 128><<<grid, kThreads, 0, st>>>(ga);
    if ((err = cudaGetLastError()) != cudaSuccess) return fail(NB_ECUDA);
    UpdateArgs u;
    u.acc64 = nullptr; u.src = d->scratch; u.acc_out = reinterpret_cast<float4*>(acc);
    u.posm = nullptr; u.vel = nullptr; u.dev = nullptr;      // no kick, no drift, no step count: untouched
    u.n = (int)n; u.nsrc = p.nsplit; u.kick_h = 0.f; u.drift_dt = 0.f; u.vscale = 1.f; u.advance = 0;
    nb_reduce_update_kernel<<<(int)((n + 255) / 256), 256, 0, st>>>(u);
    if ((err = cudaGetLastError()) != cudaSuccess) return fail(NB_ECUDA);
    return NB_OK;
}

}  // extern "C"
