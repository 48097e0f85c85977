// nb_kernels.cuh -- sm_100a kernels of the all-pairs binary-star element model.
//
// Hot path:
//   a2     nb_gravity_sym_kernel    all-pairs Eq. 4 gravity, every unordered pair once
//          nb_gravity_kernel        the same sum over every ordered pair (small and very large n)
//   a3     nb_contact_cell_kernel   contact terms of Eqs. 5/6 for exactly the
//                                   pairs with r < R_i + R_j, found through a cell list (nb_cells.cuh);
//          nb_contact_chunk_kernel  the same for n < 8,192, every pair pre-tested
//   a4/a6  nb_reduce_update_kernel  partial-sum reduction fused with the leapfrog kick/drift and
//                                   the expanding-star rule
//   a7     nb_potential_kernel / nb_moments_kernel   diagnostics for nb_energy
//
// The gravity kernel is bound by the plain FP32 ALUs (FMA pipe; register-file read bandwidth
// and the XU pipe close behind): per interaction 13.5 FP32 operations issued as packed
// FFMA2/FADD2/FMUL2, one MUFU.RSQ and half a MUFU.RCP.  Not a dense contraction: no tensor cores.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nb {

constexpr int kThreads = 128;          // 4 warps: one per SM sub-partition
constexpr float kTinyR2 = 1.0e-18f;    // added to r^2: keeps the self pair (d = 0) finite even for eps = 0,
                                       // and t0*t1 of a Montgomery pair above the fp32 normal range
constexpr float kFarAway = 1.0e10f;    // padding elements sit here with zero mass

// Device-resident mutable state (head of the workspace); updated on the device so
// that a sequence of steps needs no host round trip (graph-safe).
struct DevState {
    long long step;        // n: leapfrog steps taken since nb_set_state
    float R[2];            // element radius per star at step n (expanding-star rule)
    int n1;                // number of star-0 elements (validated)
    int bad;               // star[] validation: non-zero if not 0...0 1...1
    double R_start[2], R_end[2];
    long long n_ramp;
    long long pad_[2];
};

__device__ __forceinline__ float rsqrt_approx(float x) {
    float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y;
}

// Packed FP32 (sm_100 FFMA2/FADD2/FMUL2): two fp32 lanes in a 64-bit register pair,
// one issue slot for two operations.  ptxas folds pk2(s, s) of a scalar into a
// broadcast operand (R.F32), so tile data and constants need no duplication.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) {
    f32x2 d; asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi)); return d;
}
__device__ __forceinline__ void unpk2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d;
}

// Packed operations that the compiler may neither reorder among themselves nor fold (see sym_step).
__device__ __forceinline__ f32x2 fma2v(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d;
}

// Radius of the star an element index belongs to (star 0 first, then star 1).
__device__ __forceinline__ float star_radius(int idx, int n1, float R0, float R1) {
    return idx < n1 ? R0 : R1;
}

// ---------------------------------------------------------------------------
// Row a2: all-pairs gravity, Eq. 4, one CTA per (i-block, j-split).
//
//   a_i += G m_j / (r + eps)^2 * d/r,   d = x_j - x_i,  every j (the self pair has d = 0)
//
// Each thread keeps I (even) elements i in registers as I/2 packed pairs; the CTA
// streams its j range through shared memory in tiles of TJ elements (double-buffered,
// one barrier per tile); every LDS.128 of (x_j, y_j, z_j, G m_j) is a warp broadcast.
// Per packed lane pair and TWO elements j the loop issues
//     FADD2 x6 (d), FFMA2 x6 (r^2), MUFU.RSQ x4 (y = 1/r), FFMA2 x2 (s = r^2 y + eps),
//     FMUL2 x2 (t = s^2), FMUL2 (P = t0 t1), MUFU.RCP x2 (1/P), FMUL2 x2 (k0 = t1 y0, k1 = t0 y1),
//     FMUL2 x2 (c = k/P = y/t), FFMA2 x6 (a += c d)
// i.e. 13.5 packed FP32 instructions and 1.5 MUFU per interaction: the reciprocal of
// (r+eps)^2 is shared by the two j of a lane (Montgomery's trick: 1/t0 = t1/(t0 t1)), entirely
// in packed form.  t >= max(eps^2, kTinyR2) so the product cannot underflow; a padding element
// (1e10 away) overflows P to +inf -> 1/P = 0 -> contributes exactly 0.
// Tiles whose elements all have the same mass (the paper's stars are made of equal-mass
// elements) skip the per-pair multiply by G m_j: the tile's fp32 sums are
// scaled once when they are flushed into the fp64 accumulators.  Other tiles multiply k by
// G m_j (one more FMUL2 per lane pair and j).
// (No __restrict__ on these members: nb_fused_step_kernel writes the same arrays in another phase of the same
// launch, and loads through the read-only path would then be undefined.)
struct GravArgs {
    const float4* posm;                // [n] x,y,z,m
    float4* part;                      // [nsplit][n] partial accelerations
    int n, nib, nsplit, njt;
    float G, eps;
};

constexpr int kGroupJ = 4;             // elements j per unrolled group (two Montgomery pairs)

// Contact terms found INSIDE the all-pairs loop (CON = true: the fused small-n kernel, where a separate contact
// pass would be one more chain of latencies; the big kernels keep the test out of the loop, see 5.1b of DESIGN.md).
struct ContactArgs;
__device__ __forceinline__ void contact_pair(const ContactArgs& a, const float4 pi, const float4 vi, const float4 pj,
                                             const float4 vj, double& fx, double& fy, double& fz);
constexpr int kInlineQueue = 24;       // per-thread queue of (i slot, j) pairs that passed the fp32 pre-test
struct InlineContact {
    const ContactArgs* law;            // gamma, gamma_beta, v_dead, lens_mode
    const float4* vel;                 // [n]
    int n1;
    float R0, R1;                      // element radius per star
    uint32_t* q;                       // the thread's queue: q[k * kThreads], k < kInlineQueue
    int* pre;                          // [kThreads / 32][33]  scratch of the warp-balanced evaluation
    double* res;                       // [kThreads / 32][kInlineRound][3]
};
constexpr int kInlineRound = 64;       // pairs a warp evaluates per round

template <int H, bool UNI, bool CON>
__device__ __forceinline__ void gravity_group(const float4* __restrict__ s,
                                              const f32x2 (&nxi)[H], const f32x2 (&nyi)[H], const f32x2 (&nzi)[H],
                                              f32x2 eps2, f32x2 (&ax)[H], f32x2 (&ay)[H], f32x2 (&az)[H],
                                              const float thr, const int jglob, uint32_t* __restrict__ q, int& nq)
{
    const f32x2 tiny2 = pk2(kTinyR2, kTinyR2);
#pragma unroll
    for (int u = 0; u < kGroupJ; u += 2) {
        const float4 p0 = s[u], p1 = s[u + 1];                     // LDS.128 broadcasts
        const f32x2 x0 = pk2(p0.x, p0.x), y0 = pk2(p0.y, p0.y), z0 = pk2(p0.z, p0.z);
        const f32x2 x1 = pk2(p1.x, p1.x), y1 = pk2(p1.y, p1.y), z1 = pk2(p1.z, p1.z);
#pragma unroll
        for (int h = 0; h < H; ++h) {
            const f32x2 dx0 = add2(x0, nxi[h]), dy0 = add2(y0, nyi[h]), dz0 = add2(z0, nzi[h]);
            const f32x2 dx1 = add2(x1, nxi[h]), dy1 = add2(y1, nyi[h]), dz1 = add2(z1, nzi[h]);
            f32x2 r20 = fma2(dx0, dx0, tiny2); r20 = fma2(dy0, dy0, r20); r20 = fma2(dz0, dz0, r20);
            f32x2 r21 = fma2(dx1, dx1, tiny2); r21 = fma2(dy1, dy1, r21); r21 = fma2(dz1, dz1, r21);
            float a0, b0, a1, b1;
            unpk2(r20, a0, b0); unpk2(r21, a1, b1);
            if (CON) {                               // within reach of a contact (or the self pair): queue for the fp64 test
                if (fminf(fminf(a0, b0), fminf(a1, b1)) <= thr) {
                    const uint32_t j0 = (uint32_t)(jglob + u), sl = (uint32_t)(2 * h);
                    if (a0 <= thr) q[(nq++) * kThreads] = (j0 << 4) | sl;
                    if (b0 <= thr) q[(nq++) * kThreads] = (j0 << 4) | (sl + 1);
                    if (a1 <= thr) q[(nq++) * kThreads] = ((j0 + 1) << 4) | sl;
                    if (b1 <= thr) q[(nq++) * kThreads] = ((j0 + 1) << 4) | (sl + 1);
                }
            }
            const f32x2 ri0 = pk2(rsqrt_approx(a0), rsqrt_approx(b0));     // 1/r
            const f32x2 ri1 = pk2(rsqrt_approx(a1), rsqrt_approx(b1));
            const f32x2 s0 = fma2(r20, ri0, eps2), s1 = fma2(r21, ri1, eps2);   // r + eps
            const f32x2 t0 = mul2(s0, s0), t1 = mul2(s1, s1);                   // (r + eps)^2
            const f32x2 P = mul2(t0, t1);
            float pl, ph;
            unpk2(P, pl, ph);
            const f32x2 iP = pk2(rcp_approx(pl), rcp_approx(ph));              // one RCP per two interactions
            f32x2 k0 = mul2(t1, ri0), k1 = mul2(t0, ri1);
            if (!UNI) { k0 = mul2(k0, pk2(p0.w, p0.w)); k1 = mul2(k1, pk2(p1.w, p1.w)); }   // G m_j
            const f32x2 c0 = mul2(iP, k0), c1 = mul2(iP, k1);                  // [G m_j]/(r (r+eps)^2)  Eq. 4
            ax[h] = fma2(c0, dx0, ax[h]); ay[h] = fma2(c0, dy0, ay[h]); az[h] = fma2(c0, dz0, az[h]);
            ax[h] = fma2(c1, dx1, ax[h]); ay[h] = fma2(c1, dy1, ay[h]); az[h] = fma2(c1, dz1, az[h]);
        }
    }
}

// The work of one CTA (i-block, j-split) = block `vb` of a grid of nib * nsplit; sj: the CTA's two tiles.
template <int I, int TJ, bool CON = false>
__device__ __forceinline__ void gravity_block(const GravArgs& a, const int vb, float4 (*sj)[TJ],
                                              const InlineContact ic = InlineContact())
{
    static_assert(I % 2 == 0 && TJ % kThreads == 0 && TJ % kGroupJ == 0, "packed pairs; whole groups");
    static_assert(I <= 16 && kInlineQueue >= 2 * kGroupJ * I, "queue entries carry the i slot in 4 bits; a group adds <= 4 I");
    constexpr int H = I / 2;                        // packed pairs per thread
    constexpr int LPT = TJ / kThreads;              // tile loads per thread

    const int tid = threadIdx.x;
    const int ib = vb % a.nib;
    const int sp = vb / a.nib;
    const int ibase = ib * (kThreads * I) + tid;    // element k of this thread: ibase + k*kThreads

    f32x2 nxi[H], nyi[H], nzi[H];                   // (-x_i) of the two lanes
#pragma unroll
    for (int h = 0; h < H; ++h) {
        float px[2], py[2], pz[2];
#pragma unroll
        for (int l = 0; l < 2; ++l) {
            const int i = ibase + (2 * h + l) * kThreads;
            if (i < a.n) {
                const float4 p = a.posm[i];
                px[l] = -p.x; py[l] = -p.y; pz[l] = -p.z;
            } else {
                px[l] = py[l] = pz[l] = kFarAway;
            }
        }
        nxi[h] = pk2(px[0], px[1]); nyi[h] = pk2(py[0], py[1]); nzi[h] = pk2(pz[0], pz[1]);
    }

    const int t0 = (int)(((long long)sp * a.njt) / a.nsplit);
    const int t1 = (int)(((long long)(sp + 1) * a.njt) / a.nsplit);

    double accx[I], accy[I], accz[I];
#pragma unroll
    for (int k = 0; k < I; ++k) accx[k] = accy[k] = accz[k] = 0.0;

    // inline contact search: one fp32 threshold per thread and tile, (largest R_i of the thread's elements +
    // largest R_j of the tile)^2 -- tiles rarely straddle the two stars, so this is the pair's own reach
    float thr = -1.f, Rm = 0.f;
    int nq = 0;
    uint32_t* __restrict__ q = ic.q;
    if (CON) {
#pragma unroll
        for (int k = 0; k < I; ++k) Rm = fmaxf(Rm, star_radius(min(ibase + k * kThreads, a.n - 1), ic.n1, ic.R0, ic.R1));
    }
    // what contact_pair() needs of the thread's own elements: (x, R) and (v, m); x_j comes from the tile in shared
    // memory, so a queued pair costs ONE global load (v_j)
    float4 cpi[CON ? I : 1], cvi[CON ? I : 1];
    if (CON) {
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const int i = min(ibase + k * kThreads, a.n - 1);
            const float4 x = a.posm[i], w = ic.vel[i];
            cpi[k] = make_float4(x.x, x.y, x.z, star_radius(i, ic.n1, ic.R0, ic.R1));
            cvi[k] = make_float4(w.x, w.y, w.z, x.w);
        }
    }
    const float4* tile = nullptr;                    // the tile being walked, and the index of its first element
    int tile_j0 = 0;
    auto drain = [&]() {                             // the queued pairs, in the order found, in fp64
        for (int e0 = 0; e0 < nq; e0 += 2) {
            int jj[2], kk[2];
            float4 wj[2];
            bool ok[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {            // both loads in flight together
                const uint32_t w = q[min(e0 + u, nq - 1) * kThreads];
                jj[u] = (int)(w >> 4); kk[u] = (int)(w & 15u);
                ok[u] = e0 + u < nq && jj[u] < a.n && ibase + kk[u] * kThreads < a.n && jj[u] != ibase + kk[u] * kThreads;
                wj[u] = ok[u] ? ic.vel[jj[u]] : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                if (!ok[u]) continue;
                const float4 xj = tile[jj[u] - tile_j0];
                float4 pi = cpi[0], vi = cvi[0];
#pragma unroll
                for (int k = 1; k < I; ++k) if (k == kk[u]) { pi = cpi[k]; vi = cvi[k]; }
                double fx, fy, fz;
                contact_pair(*ic.law, pi, vi, make_float4(xj.x, xj.y, xj.z, star_radius(jj[u], ic.n1, ic.R0, ic.R1)), wj[u],
                             fx, fy, fz);
                const double im = 1.0 / (double)vi.w;
#pragma unroll
                for (int k = 0; k < I; ++k)
                    if (k == kk[u]) { accx[k] += fx * im; accy[k] += fy * im; accz[k] += fz * im; }
            }
        }
        nq = 0;
    };

    // The same at a point where the whole warp arrives together (the end of a tile): the warp's queued pairs are
    // dealt evenly to its lanes -- a lane with 6 pairs no longer holds up 31 lanes with 1 -- evaluated, and handed
    // back through shared memory; every lane adds up ITS pairs in the order it found them.
    auto drain_warp = [&]() {
        const int lane = tid & 31, wq = tid >> 5;
        int inc = nq;
        for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
        const int total = __shfl_sync(0xffffffffu, inc, 31), mine0 = inc - nq;
        int* pre = ic.pre + wq * 33;
        double* res = ic.res + wq * (kInlineRound * 3);
        pre[lane] = mine0;
        if (lane == 31) pre[32] = total;
        __syncwarp();
        for (int p0 = 0; p0 < total; p0 += kInlineRound) {
            const int pe = min(total, p0 + kInlineRound);
            for (int p = p0 + lane; p < pe; p += 32) {
                int lo = 0;                          // owner: the largest lane with pre[lane] <= p
#pragma unroll
                for (int s2 = 16; s2 > 0; s2 >>= 1) if (pre[lo + s2] <= p) lo += s2;
                const uint32_t w = (q - lane)[(p - pre[lo]) * kThreads + lo];
                const int j = (int)(w >> 4), i = ibase - lane + lo + (int)(w & 15u) * kThreads;
                double fx = 0.0, fy = 0.0, fz = 0.0;
                if (j < a.n && i < a.n && j != i) {
                    const float4 xi = a.posm[i], wi = ic.vel[i], wj = ic.vel[j], xj = tile[j - tile_j0];
                    contact_pair(*ic.law, make_float4(xi.x, xi.y, xi.z, star_radius(i, ic.n1, ic.R0, ic.R1)),
                                 make_float4(wi.x, wi.y, wi.z, xi.w),
                                 make_float4(xj.x, xj.y, xj.z, star_radius(j, ic.n1, ic.R0, ic.R1)), wj, fx, fy, fz);
                    const double im = 1.0 / (double)xi.w;
                    fx *= im; fy *= im; fz *= im;
                }
                res[(p - p0) * 3] = fx; res[(p - p0) * 3 + 1] = fy; res[(p - p0) * 3 + 2] = fz;
            }
            __syncwarp();
            const int b = max(mine0, p0), e = min(mine0 + nq, pe);
            for (int p = b; p < e; ++p) {
                const int k = (int)(q[(p - mine0) * kThreads] & 15u);
#pragma unroll
                for (int kk = 0; kk < I; ++kk)
                    if (kk == k) { accx[kk] += res[(p - p0) * 3]; accy[kk] += res[(p - p0) * 3 + 1]; accz[kk] += res[(p - p0) * 3 + 2]; }
            }
            __syncwarp();
        }
        nq = 0;
    };

    float4 pre[LPT];
    bool my_uni = false;                             // this thread's share of the tile has one mass
    auto load_tile = [&](int t) {
        const float mref = a.posm[min(t * TJ, a.n - 1)].w;
        bool u = true;
#pragma unroll
        for (int l = 0; l < LPT; ++l) {
            const int j = t * TJ + l * kThreads + tid;
            if (j < a.n) {
                pre[l] = a.posm[j];
                u = u && (pre[l].w == mref);
                pre[l].w *= a.G;                                   // fold G into m_j
            } else {
                pre[l] = make_float4(kFarAway, kFarAway, kFarAway, 0.f);
                u = false;
            }
        }
        my_uni = u;
    };
    auto store_tile = [&](int buf) {
#pragma unroll
        for (int l = 0; l < LPT; ++l) sj[buf][l * kThreads + tid] = pre[l];
    };

    if (t0 < t1) { load_tile(t0); store_tile(0); }
    int uni = __syncthreads_and(my_uni ? 1 : 0);

    const f32x2 eps2 = pk2(a.eps, a.eps);

    for (int t = t0; t < t1; ++t) {
        const int buf = (t - t0) & 1;
        if (t + 1 < t1) load_tile(t + 1);            // global loads overlap the tile's math

        f32x2 ax[H], ay[H], az[H];
#pragma unroll
        for (int h = 0; h < H; ++h) ax[h] = ay[h] = az[h] = pk2(0.f, 0.f);

        const float4* __restrict__ s = sj[buf];
        tile = s; tile_j0 = t * TJ;
        if (CON) {
            const float Rj = (t + 1) * TJ <= ic.n1 ? ic.R0 : (t * TJ >= ic.n1 ? ic.R1 : fmaxf(ic.R0, ic.R1));
            const float D = Rm + Rj;
            thr = D * D * (1.0f + 1.0e-5f) + kTinyR2;
        }
        double scale = 1.0;
        if (uni) {
#pragma unroll 1
            for (int jg = 0; jg < TJ; jg += kGroupJ) {
                gravity_group<H, true, CON>(s + jg, nxi, nyi, nzi, eps2, ax, ay, az, thr, t * TJ + jg, q, nq);
                if (CON && nq > kInlineQueue - 2 * kGroupJ * H) drain();
            }
            scale = (double)s[0].w;                  // G m of the whole tile
        } else {
#pragma unroll 1
            for (int jg = 0; jg < TJ; jg += kGroupJ) {
                gravity_group<H, false, CON>(s + jg, nxi, nyi, nzi, eps2, ax, ay, az, thr, t * TJ + jg, q, nq);
                if (CON && nq > kInlineQueue - 2 * kGroupJ * H) drain();
            }
        }
        if (CON) drain_warp();

        // flush the tile's fp32 sums into the fp64 accumulators (short fp32 chains)
#pragma unroll
        for (int h = 0; h < H; ++h) {
            float l, hgh;
            unpk2(ax[h], l, hgh); accx[2 * h] += scale * (double)l; accx[2 * h + 1] += scale * (double)hgh;
            unpk2(ay[h], l, hgh); accy[2 * h] += scale * (double)l; accy[2 * h + 1] += scale * (double)hgh;
            unpk2(az[h], l, hgh); accz[2 * h] += scale * (double)l; accz[2 * h + 1] += scale * (double)hgh;
        }

        if (t + 1 < t1) store_tile(buf ^ 1);
        uni = __syncthreads_and(my_uni ? 1 : 0);
    }

    float4* __restrict__ out = a.part + (size_t)sp * a.n;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = ibase + k * kThreads;
        if (i < a.n) out[i] = make_float4((float)accx[k], (float)accy[k], (float)accz[k], 0.f);
    }
}

template <int I, int TJ>
__global__ void __launch_bounds__(kThreads, (I == 2 ? 8 : 4))
nb_gravity_kernel(const __grid_constant__ GravArgs a)
{
    __shared__ float4 sj[2][TJ];
    gravity_block<I, TJ>(a, blockIdx.x, sj);
}

// ---------------------------------------------------------------------------
// Row a2 for large N: the same sum with every UNORDERED pair evaluated once.
//
// Eq. 4 is a force "between elements i and j": F_ij = -F_ji, so the geometric
// factor c = 1/(r (r+eps)^2) and the difference d of a pair serve both a_i += G m_j c d and
// a_j -= G m_i c d.  Elements are cut into super-tiles of S; one CTA owns one pair of
// super-tiles (A <= B) and stages B in shared memory as PACKED PAIRS: pair p of tile t holds
// elements 64 t + p and 64 t + 32 + p (float2 arrays X2, Y2, Z2, M2).  Each of its NT/32 warps
// keeps 32 NI elements i of A in registers (NI per lane, as broadcast scalars) and walks the
// tiles of B.  Inside a tile the warp ROTATES: at step k lane l meets pair (l+k)&31 (three
// conflict-free LDS.64), so both accumulations are lane-aligned packed FFMA2 with the same
// sources (c, d):  a_i += c d  into a per-i accumulator whose halves are the sums over the two
// slot families (added once per round), and the reaction  a_j += c d  into one packed register
// triple that TRAVELS WITH THE PAIR (SHFL to lane l-1 after every step).  The two FFMA2 are issued
// back to back (asm volatile keeps the order): the second takes (c, d) from the operand reuse
// cache and reads only its accumulator from the register file.  After 32 steps the lane holds the
// finished reaction sums of pair l over the warp's 32 NI elements i and adds them to the CTA's
// shared-memory array.  The warps of a CTA are skewed over different tiles and meet at a barrier
// after every tile, so the shared-memory sums have a fixed order: bitwise reproducible.
// Per lane and step at NI = 8 (8 i x 2 j = 16 pairs = 32 interactions): 120 packed FP32 instructions
// (FADD2 x24, FFMA2 x24+8, FMUL2 x16, FFMA2 x24+24), 32 MUFU (one RSQ and one RCP per pair: a pair
// evaluation already serves two interactions, so the shared reciprocal of the one-sided kernel
// would cost more FMA-pipe cycles than the XU cycles it saves), 6 SHFL, 3 LDS.64 -- 13.5 executed
// flop per interaction against 22 one-sided.  DESIGN.md 5.1c lists the variants measured on the way
// (packed lanes along i with horizontal adds, Montgomery, NI, CTA shapes, unrolls).
// Output: part[Y][e] = acceleration of element e due to the elements of super-tile Y (every
// (Y, tile of e) combination is written by exactly one CTA; the diagonal CTAs (A == B) run the
// one-sided loop).  Super-tiles of one mass take the mass out of the loop, as in
// the one-sided kernel; other pairs of super-tiles multiply c by G m_j and G m_i per pair.
// Template parameters: S super-tile, NI elements i per lane, NT threads, MINB CTAs/SM, UNR unroll
// of the 32-step rotation (shipped: 8 i per lane, 128 threads, 2 CTAs/SM, unroll 16 at S >= 512: 254 registers,
// 8 warps per SM).  A step is written phase by phase over the NI elements i
// (d and r^2 of all, then all MUFU.RSQ, ...), which keeps the MUFU of all of them in flight together.
struct SymArgs {
    const float4* __restrict__ posm;   // [n] x,y,z,m
    float4* __restrict__ part;         // [T][n]   (slab mode)
    double* __restrict__ acc64;        // [6][n]   (chain mode) a_i side x,y,z then reaction side x,y,z
    int* __restrict__ turn;            // (chain mode) turnA[T rounds], turnR[T], ticket, error flag -- zero at launch
    int n, T;                          // T = ceil(n / S) super-tiles
    float G, eps;
};

// Chain mode (n >= 98,304): instead of T slabs of partial sums -- 1.1 GB at N = 262,144, 5 GB at 1,048,576 --
// the CTAs add their results straight into ONE pair of fp64 accumulators per element, each super-tile's
// contributions in a fixed order enforced by a turn counter per tile: bitwise reproducible, no atomics on data.
// A CTA takes a ticket when it STARTS (so every lower ticket belongs to a CTA that is resident or done -- the
// forward-progress argument of a decoupled look-back scan) and the tickets walk the pairs of super-tiles in
// DIAGONAL-MAJOR order (d = B - A = 0, 1, 2, ...): the a_i side of (A, B) goes to tile A at turn d, after
// (A, B-1); its reaction goes to tile B at turn d-1, after (A+1, B) -- both predecessors lie on the previous
// diagonal, i.e. hold lower tickets, taken ~T tickets (a whole wave of CTAs) earlier: a CTA finds that its turn
// has come when it gets there, the waits cost nothing, and no CTA ever waits for a higher ticket.
__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v; asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
    asm volatile("st.release.gpu.global.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
constexpr int kChainSpinLimit = 1 << 22;     // x 100 ns: ~0.4 s, then the error flag is raised and the CTA goes on

// Block-wide: wait until *turn == want (thread 0 polls; a lost turn raises *err instead of hanging the GPU).
__device__ __forceinline__ void chain_wait(int* turn, int want, int* err) {
    if (threadIdx.x == 0) {
        int spins = 0;
        while (ld_acquire_gpu(turn) != want) {
            __nanosleep(100);
            if (++spins > kChainSpinLimit) { atomicExch(err, 1); break; }
        }
    }
    __syncthreads();
}
// Block-wide: publish the block's accumulator updates and pass the turn on.  The barrier orders the other
// threads' stores before thread 0's release, which is cumulative: no fence per thread.
__device__ __forceinline__ void chain_release(int* turn, int next) {
    __syncthreads();
    if (threadIdx.x == 0) st_release_gpu(turn, next);
}

constexpr int kSymSmemPerElem = 28;    // dynamic shared memory of the symmetric kernel: (16 + 3*4) bytes x S

#ifndef NB_SYM_GROUP
#define NB_SYM_GROUP 8       // elements i whose phases are interleaved (all d and r^2, then all MUFU.RSQ, ...)
#endif

template <int NI, bool UNI, bool SYM>
__device__ __forceinline__ void sym_step(const f32x2 X, const f32x2 Y, const f32x2 Z, const f32x2 M,
                                         const float (&nxi)[NI], const float (&nyi)[NI], const float (&nzi)[NI],
                                         const float (&gmi)[NI], const f32x2 eps2,
                                         f32x2 (&ax)[NI], f32x2 (&ay)[NI], f32x2 (&az)[NI],
                                         f32x2& jx, f32x2& jy, f32x2& jz)
{
    constexpr int GI = NI < NB_SYM_GROUP ? NI : NB_SYM_GROUP;
    static_assert(NI % GI == 0, "whole groups of elements i");
    const f32x2 tiny2 = pk2(kTinyR2, kTinyR2);
#pragma unroll
    for (int g = 0; g < NI; g += GI) {
        f32x2 dx[GI], dy[GI], dz[GI], r2[GI], ri[GI], t[GI], c[GI];
        // phase by phase over the GI elements i, so that the MUFU of all of them are in flight together
#pragma unroll
        for (int i = 0; i < GI; ++i) {
            dx[i] = add2(X, pk2(nxi[g + i], nxi[g + i])); dy[i] = add2(Y, pk2(nyi[g + i], nyi[g + i]));
            dz[i] = add2(Z, pk2(nzi[g + i], nzi[g + i]));
            r2[i] = fma2(dx[i], dx[i], tiny2); r2[i] = fma2(dy[i], dy[i], r2[i]); r2[i] = fma2(dz[i], dz[i], r2[i]);
        }
#pragma unroll
        for (int i = 0; i < GI; ++i) {
            float a0, b0;
            unpk2(r2[i], a0, b0);
            ri[i] = pk2(rsqrt_approx(a0), rsqrt_approx(b0));                   // 1/r
        }
#pragma unroll
        for (int i = 0; i < GI; ++i) {
            const f32x2 sm = fma2(r2[i], ri[i], eps2);                         // r + eps
            t[i] = mul2(sm, sm);                                               // (r + eps)^2
        }
#pragma unroll
        for (int i = 0; i < GI; ++i) {
            float a0, b0;
            unpk2(t[i], a0, b0);
            c[i] = mul2(ri[i], pk2(rcp_approx(a0), rcp_approx(b0)));           // 1/(r (r+eps)^2)   Eq. 4
        }
#pragma unroll
        for (int i = 0; i < GI; ++i) {
            if (UNI) {
                if (SYM) {
                    ax[g + i] = fma2v(c[i], dx[i], ax[g + i]); jx = fma2v(c[i], dx[i], jx);
                    ay[g + i] = fma2v(c[i], dy[i], ay[g + i]); jy = fma2v(c[i], dy[i], jy);
                    az[g + i] = fma2v(c[i], dz[i], az[g + i]); jz = fma2v(c[i], dz[i], jz);
                } else {
                    ax[g + i] = fma2(c[i], dx[i], ax[g + i]); ay[g + i] = fma2(c[i], dy[i], ay[g + i]);
                    az[g + i] = fma2(c[i], dz[i], az[g + i]);
                }
            } else {
                const f32x2 ci = mul2(c[i], M);                                // G m_j for a_i
                ax[g + i] = fma2(ci, dx[i], ax[g + i]); ay[g + i] = fma2(ci, dy[i], ay[g + i]);
                az[g + i] = fma2(ci, dz[i], az[g + i]);
                if (SYM) {
                    const f32x2 cj = mul2(c[i], pk2(gmi[g + i], gmi[g + i]));  // G m_i for a_j
                    jx = fma2(cj, dx[i], jx); jy = fma2(cj, dy[i], jy); jz = fma2(cj, dz[i], jz);
                }
            }
        }
    }
}

template <int S, int NI, int NT, int UNR, bool UNI, bool SYM, bool CHAIN = false>
__device__ __forceinline__ void sym_sweep(const SymArgs& a, const int A, const int B,
                                           const float2* __restrict__ X2, const float2* __restrict__ Y2,
                                           const float2* __restrict__ Z2, const float2* __restrict__ M2,
                                           float2* __restrict__ JX, float2* __restrict__ JY, float2* __restrict__ JZ,
                                           const double scale_i)
{
    constexpr int NW = NT / 32;
    constexpr int NJT = S / 64;                      // tiles of 64 elements j = 32 packed pairs
    constexpr int SKEW = NJT / NW;
    constexpr int IPR = NW * 32 * NI;                // elements i per round
    static_assert(S % (64 * NW) == 0 && S % IPR == 0, "every warp needs its own tile at every step");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int src = (lane + 1) & 31;
    const f32x2 eps2 = pk2(a.eps, a.eps);
    float4* __restrict__ out = a.part + (size_t)B * a.n;

#pragma unroll 1
    for (int r = 0; r < S / IPR; ++r) {
        const int ibase = A * S + r * IPR + warp * (32 * NI) + lane;
        float nxi[NI], nyi[NI], nzi[NI], gmi[NI];
        f32x2 ax[NI], ay[NI], az[NI];
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            const int e = ibase + i * 32;
            float4 q = make_float4(kFarAway, kFarAway, kFarAway, 0.f);
            if (e < a.n) q = a.posm[e];
            nxi[i] = -q.x; nyi[i] = -q.y; nzi[i] = -q.z; gmi[i] = a.G * q.w;
            ax[i] = ay[i] = az[i] = pk2(0.f, 0.f);
        }
#pragma unroll 1
        for (int q = 0; q < NJT; ++q) {
            const int tile = (q + warp * SKEW) & (NJT - 1);
            const int tb = tile * 32;
            f32x2 jx = pk2(0.f, 0.f), jy = jx, jz = jx;
#pragma unroll UNR
            for (int k = 0; k < 32; ++k) {
                const int slot = tb + ((lane + k) & 31);
                const f32x2 X = *reinterpret_cast<const f32x2*>(X2 + slot), Y = *reinterpret_cast<const f32x2*>(Y2 + slot),
                            Z = *reinterpret_cast<const f32x2*>(Z2 + slot);
                f32x2 M = 0;
                if (!UNI) M = *reinterpret_cast<const f32x2*>(M2 + slot);
                sym_step<NI, UNI, SYM>(X, Y, Z, M, nxi, nyi, nzi, gmi, eps2, ax, ay, az, jx, jy, jz);
                if (SYM) {
                    float l, h;
                    unpk2(jx, l, h); jx = pk2(__shfl_sync(0xffffffffu, l, src), __shfl_sync(0xffffffffu, h, src));
                    unpk2(jy, l, h); jy = pk2(__shfl_sync(0xffffffffu, l, src), __shfl_sync(0xffffffffu, h, src));
                    unpk2(jz, l, h); jz = pk2(__shfl_sync(0xffffffffu, l, src), __shfl_sync(0xffffffffu, h, src));
                }
            }
            if (SYM) {                               // after 32 rotations lane l holds the pair of slots l, 32+l
                float l, h;
                float2 v;
                v = JX[tb + lane]; unpk2(jx, l, h); v.x += l; v.y += h; JX[tb + lane] = v;
                v = JY[tb + lane]; unpk2(jy, l, h); v.x += l; v.y += h; JY[tb + lane] = v;
                v = JZ[tb + lane]; unpk2(jz, l, h); v.x += l; v.y += h; JZ[tb + lane] = v;
                __syncthreads();                     // fixed order of the shared-memory sums
            }
        }
        // chain mode: the turn counters of tile A are per ROUND (sub-tile of IPR elements), so that a pair of
        // super-tiles with several rounds hands each of them on as soon as it is done
        int* turnA = a.turn + (A * (S / IPR) + r);
        if (CHAIN) chain_wait(turnA, B - A, a.turn + a.T * (S / IPR + 1) + 1);        // after round r of (A, B-1)
        double vx[NI], vy[NI], vz[NI];
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            float xl, xh, yl, yh, zl, zh;
            unpk2(ax[i], xl, xh); unpk2(ay[i], yl, yh); unpk2(az[i], zl, zh);
            vx[i] = scale_i * ((double)xl + (double)xh); vy[i] = scale_i * ((double)yl + (double)yh);
            vz[i] = scale_i * ((double)zl + (double)zh);
        }
        if (CHAIN) {
            const size_t n = (size_t)a.n;
            if (A != B) {                            // all loads in flight together, then all stores (turn 0 stores only)
#pragma unroll
                for (int i = 0; i < NI; ++i) {
                    const int e = ibase + i * 32;
                    if (e < a.n) { vx[i] += __ldcg(a.acc64 + e); vy[i] += __ldcg(a.acc64 + n + e); vz[i] += __ldcg(a.acc64 + 2 * n + e); }
                }
            }
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                const int e = ibase + i * 32;
                if (e < a.n) { __stcg(a.acc64 + e, vx[i]); __stcg(a.acc64 + n + e, vy[i]); __stcg(a.acc64 + 2 * n + e, vz[i]); }
            }
            chain_release(turnA, B - A + 1);
        } else {
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                const int e = ibase + i * 32;
                if (e < a.n) out[e] = make_float4((float)vx[i], (float)vy[i], (float)vz[i], 0.f);
            }
        }
    }
}

// One pair of super-tiles (A <= B): stage B, sweep A's elements over it, write or chain the two results.
template <int S, int NI, int NT, int UNR, bool CHAIN>
__device__ __forceinline__ void sym_tile_pair(const SymArgs& a, const int A, const int B, float4* sym_smem)
{
    float2* __restrict__ X2 = reinterpret_cast<float2*>(sym_smem);      // 7 arrays of S/2 float2 = 28 S bytes
    float2* __restrict__ Y2 = X2 + S / 2;
    float2* __restrict__ Z2 = Y2 + S / 2;
    float2* __restrict__ M2 = Z2 + S / 2;
    float2* __restrict__ JX = M2 + S / 2;
    float2* __restrict__ JY = JX + S / 2;
    float2* __restrict__ JZ = JY + S / 2;
    const int tid = threadIdx.x;

    // stage super-tile B as packed pairs: pair p of tile t holds elements 64 t + p and 64 t + 32 + p
    const float mB = a.posm[min(B * S, a.n - 1)].w, mA = a.posm[min(A * S, a.n - 1)].w;
    bool u = true;
    for (int p = tid; p < S / 2; p += NT) {
        const int e0 = (p >> 5) * 64 + (p & 31), e1 = e0 + 32;
        float4 q0 = make_float4(kFarAway, kFarAway, kFarAway, 0.f), q1 = q0;
        if (B * S + e0 < a.n) { q0 = a.posm[B * S + e0]; u = u && (q0.w == mB); q0.w *= a.G; } else u = false;
        if (B * S + e1 < a.n) { q1 = a.posm[B * S + e1]; u = u && (q1.w == mB); q1.w *= a.G; } else u = false;
        if (A * S + e0 < a.n) u = u && (a.posm[A * S + e0].w == mA); else u = false;
        if (A * S + e1 < a.n) u = u && (a.posm[A * S + e1].w == mA); else u = false;
        X2[p] = make_float2(q0.x, q1.x); Y2[p] = make_float2(q0.y, q1.y); Z2[p] = make_float2(q0.z, q1.z);
        M2[p] = make_float2(q0.w, q1.w);
        JX[p] = JY[p] = JZ[p] = make_float2(0.f, 0.f);
    }
    const int uni = __syncthreads_and(u ? 1 : 0);

    if (A == B) {
        if (uni) sym_sweep<S, NI, NT, UNR, true, false, CHAIN>(a, A, B, X2, Y2, Z2, M2, JX, JY, JZ, (double)(a.G * mB));
        else     sym_sweep<S, NI, NT, UNR, false, false, CHAIN>(a, A, B, X2, Y2, Z2, M2, JX, JY, JZ, 1.0);
        if (CHAIN && A == 0) {                       // tile 0 receives no reaction at all: its sums are zero
            for (int e = tid; e < S && e < a.n; e += NT) {
                double* px = a.acc64 + 3 * (size_t)a.n + e;
                __stcg(px, 0.0); __stcg(px + a.n, 0.0); __stcg(px + 2 * (size_t)a.n, 0.0);
            }
        }
        return;
    }
    if (uni) sym_sweep<S, NI, NT, UNR, true, true, CHAIN>(a, A, B, X2, Y2, Z2, M2, JX, JY, JZ, (double)(a.G * mB));
    else     sym_sweep<S, NI, NT, UNR, false, true, CHAIN>(a, A, B, X2, Y2, Z2, M2, JX, JY, JZ, 1.0);

    const double scale_j = uni ? -(double)(a.G * mA) : -1.0;
    float4* __restrict__ outj = a.part + (size_t)A * a.n;
    constexpr int RNDS = S / (NT / 32 * 32 * NI);            // rounds per super-tile: turn counters [T RNDS] a_i side, [T] reaction
    int* turnR = a.turn + a.T * RNDS + B;
    if (CHAIN) chain_wait(turnR, B - A - 1, a.turn + a.T * (RNDS + 1) + 1);        // tile B's turn d - 1: after (A+1, B)
    constexpr int PER = (S / 2 + NT - 1) / NT;               // packed pairs per thread
    double v[PER][6];
    const size_t n = (size_t)a.n;
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int p = tid + k * NT;
        const float2 x = p < S / 2 ? JX[p] : make_float2(0.f, 0.f), y = p < S / 2 ? JY[p] : x, z = p < S / 2 ? JZ[p] : x;
        v[k][0] = scale_j * (double)x.x; v[k][1] = scale_j * (double)y.x; v[k][2] = scale_j * (double)z.x;
        v[k][3] = scale_j * (double)x.y; v[k][4] = scale_j * (double)y.y; v[k][5] = scale_j * (double)z.y;
    }
    if (CHAIN && B - A > 1) {                                // all loads in flight together (turn 0 stores only)
#pragma unroll
        for (int k = 0; k < PER; ++k) {
            const int p = tid + k * NT;
            const int e0 = B * S + (p >> 5) * 64 + (p & 31), e1 = e0 + 32;
            double* q = a.acc64 + 3 * n;
            if (p < S / 2 && e0 < a.n) { v[k][0] += __ldcg(q + e0); v[k][1] += __ldcg(q + n + e0); v[k][2] += __ldcg(q + 2 * n + e0); }
            if (p < S / 2 && e1 < a.n) { v[k][3] += __ldcg(q + e1); v[k][4] += __ldcg(q + n + e1); v[k][5] += __ldcg(q + 2 * n + e1); }
        }
    }
#pragma unroll
    for (int k = 0; k < PER; ++k) {
        const int p = tid + k * NT;
        const int e0 = B * S + (p >> 5) * 64 + (p & 31), e1 = e0 + 32;
        if (p >= S / 2) continue;
        if (CHAIN) {
            double* q = a.acc64 + 3 * n;
            if (e0 < a.n) { __stcg(q + e0, v[k][0]); __stcg(q + n + e0, v[k][1]); __stcg(q + 2 * n + e0, v[k][2]); }
            if (e1 < a.n) { __stcg(q + e1, v[k][3]); __stcg(q + n + e1, v[k][4]); __stcg(q + 2 * n + e1, v[k][5]); }
        } else {
            if (e0 < a.n) outj[e0] = make_float4((float)v[k][0], (float)v[k][1], (float)v[k][2], 0.f);
            if (e1 < a.n) outj[e1] = make_float4((float)v[k][3], (float)v[k][4], (float)v[k][5], 0.f);
        }
    }
    if (CHAIN) chain_release(turnR, B - A);
}


template <int S, int NI, int NT, int MINB, int UNR>
__global__ void __launch_bounds__(NT, MINB)
nb_gravity_sym_kernel(const __grid_constant__ SymArgs a)
{
    extern __shared__ float4 sym_smem[];
    int A, B;
    {
        const long long T = a.T, M = T * (T - 1) / 2, b = blockIdx.x;
        if (b >= M) { A = B = (int)(b - M); }
        else {
            const double t2 = 2.0 * (double)T - 1.0;
            long long r = (long long)((t2 - sqrt(t2 * t2 - 8.0 * (double)b)) * 0.5);
            if (r < 0) r = 0;
            while (r > 0 && r * (2 * T - r - 1) / 2 > b) --r;
            while ((r + 1) * (2 * T - r - 2) / 2 <= b) ++r;
            A = (int)r;
            B = (int)(b - r * (2 * T - r - 1) / 2 + r + 1);
        }
    }
    sym_tile_pair<S, NI, NT, UNR, false>(a, A, B, sym_smem);
}

// Chain mode: every CTA takes a ticket when it starts and works on that pair of super-tiles, diagonal-major.
template <int S, int NI, int NT, int MINB, int UNR>
__global__ void __launch_bounds__(NT, MINB)
nb_gravity_sym_chain_kernel(const __grid_constant__ SymArgs a)
{
    extern __shared__ float4 sym_smem[];
    __shared__ int s_ticket;
    constexpr int RNDS = S / (NT / 32 * 32 * NI);
    if (threadIdx.x == 0) s_ticket = atomicAdd(a.turn + a.T * (RNDS + 1), 1);
    __syncthreads();
    const long long T = a.T, t = s_ticket;
    // diagonal d holds T - d pairs; c(d) = d T - d (d - 1) / 2 pairs lie on the diagonals before it
    const double t2 = 2.0 * (double)T + 1.0;
    long long d = (long long)((t2 - sqrt(t2 * t2 - 8.0 * (double)t)) * 0.5);
    if (d < 0) d = 0;
    if (d > T - 1) d = T - 1;
    while (d > 0 && d * T - d * (d - 1) / 2 > t) --d;
    while (d < T - 1 && (d + 1) * T - (d + 1) * d / 2 <= t) ++d;
    const int A = (int)(t - (d * T - d * (d - 1) / 2));
    sym_tile_pair<S, NI, NT, UNR, true>(a, A, A + (int)d, sym_smem);
}

// ---------------------------------------------------------------------------
// Row a3: contact repulsion, Eqs. 5/6, for exactly the pairs with
// r < R_i + R_j.  These are ~5 pairs per element out of N, so they are found by a spatial
// search instead of a test inside the N^2 loop: for n >= 8,192 through the cell list of
// nb_cells.cuh; for smaller n (where a warp per 32 elements cannot fill the machine anyway) by
// testing every pair, dealt to many warps:
//   nb_gather_kernel        ps = (x,y,z,R_star), vs = (vx,vy,vz,m) in index order; bounding box +
//                           largest radius of every group of 32 elements
//   nb_contact_chunk_kernel one warp per (group of 32 elements i, chunk of groups j): each lane's
//                           point against the box of every group of the chunk, then every j of the
//                           groups that survive; a pair in contact is evaluated in fp64.
// The box and fp32 tests are conservative (a pair in contact is never skipped); which pairs ARE in
// contact is decided by the fp64 test r < R_i + R_j alone.
constexpr int kBoxBlocks = 128;       // blocks (= partial boxes) of nb_cell_bbox_kernel
constexpr int kGroup = 32;            // elements per group (one warp)
constexpr int kSuper = 32;            // groups per super-group (one 1024-thread block of the gather)

__device__ __forceinline__ float warp_min(float v) {
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// One 1024-thread block per super-group.  gbox[2g] = (lo.xyz, Rmax), gbox[2g+1] = (hi.xyz, 0);
// sbox likewise per block.
__global__ void __launch_bounds__(kGroup * kSuper)
nb_gather_kernel(const float4* __restrict__ posm, const float4* __restrict__ vel, const uint32_t* __restrict__ perm,
                 int n, const DevState* __restrict__ dev, float4* __restrict__ ps, float4* __restrict__ vs,
                 float4* __restrict__ gbox, float4* __restrict__ sbox)
{
    __shared__ float sh[7][kSuper];
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, rmax = 0.f;
    if (k < n) {
        const int src = perm ? (int)perm[k] : k;
        const float4 p = posm[src], v = vel[src];
        const float R = star_radius(src, dev->n1, dev->R[0], dev->R[1]);
        ps[k] = make_float4(p.x, p.y, p.z, R);
        vs[k] = make_float4(v.x, v.y, v.z, p.w);
        lo[0] = hi[0] = p.x; lo[1] = hi[1] = p.y; lo[2] = hi[2] = p.z; rmax = R;
    }
    for (int c = 0; c < 3; ++c) { lo[c] = warp_min(lo[c]); hi[c] = warp_max(hi[c]); }
    rmax = warp_max(rmax);
    const int g = blockIdx.x * kSuper + w;
    if (l == 0) {
        if ((long long)g * kGroup < n) {
            gbox[2 * g] = make_float4(lo[0], lo[1], lo[2], rmax);
            gbox[2 * g + 1] = make_float4(hi[0], hi[1], hi[2], 0.f);
        }
        for (int c = 0; c < 3; ++c) { sh[c][w] = lo[c]; sh[3 + c][w] = hi[c]; }
        sh[6][w] = rmax;
    }
    __syncthreads();
    if (w == 0) {
        float q[7];
        for (int c = 0; c < 3; ++c) { q[c] = warp_min(sh[c][l]); q[3 + c] = warp_max(sh[3 + c][l]); }
        q[6] = warp_max(sh[6][l]);
        if (l == 0) {
            sbox[2 * blockIdx.x] = make_float4(q[0], q[1], q[2], q[6]);
            sbox[2 * blockIdx.x + 1] = make_float4(q[3], q[4], q[5], 0.f);
        }
    }
}

struct ContactArgs {
    const float4* ps;                  // [n] x,y,z,R_star
    const float4* vs;                  // [n] vx,vy,vz,m
    const uint32_t* perm;              // [n] original index of sorted element k (nullptr: identity)
    const float4* gbox;                // [2*ngroups]
    const float4* sbox;                // [2*nsuper]
    float4* out;                       // [nchunks][n] contact acceleration, ORIGINAL index order
    int n, ngroups, nsuper;
    int nchunks;                       // slabs of `out` (index-order search: one per chunk of candidate groups)
    float gamma, gamma_beta;           // Eq. 5 / Eq. 6 strengths
    float v_dead;
    int lens_mode;
};

// Squared gap between two axis-aligned boxes (0 if they overlap).
__device__ __forceinline__ float box_gap2(const float4 alo, const float4 ahi, const float4 blo, const float4 bhi) {
    const float gx = fmaxf(0.f, fmaxf(alo.x - bhi.x, blo.x - ahi.x));
    const float gy = fmaxf(0.f, fmaxf(alo.y - bhi.y, blo.y - ahi.y));
    const float gz = fmaxf(0.f, fmaxf(alo.z - bhi.z, blo.z - ahi.z));
    return gx * gx + gy * gy + gz * gz;
}

// The contact term of one (i, j) pair, Eqs. 5/6, added to the fp64
// accumulators of i:  a_i -= g pi V(r; R_ij) / m_i * d/r  if 0 < r < R_i + R_j  (A2, A3).
// Evaluated in double throughout (h = 2R - r cancels badly in fp32 near first contact);
// d is the exact difference of the fp32 coordinates.
// lens_mode 0: pi V = pi (D - r)^2 (2D + r) / 12 with D = 2 R_ij (factored displaced
// volume, A1); lens_mode 1: the polynomial as printed, last term r^2/12.
__device__ __forceinline__ void contact_term(const ContactArgs& a, const float4 pi, const float4 vi,
                                             const float4 pj, const float4 vj,
                                             double& ax, double& ay, double& az)
{
    const double dx = (double)pj.x - (double)pi.x, dy = (double)pj.y - (double)pi.y, dz = (double)pj.z - (double)pi.z;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double D = (double)pi.w + (double)pj.w;                   // R_i + R_j = 2 R_ij (A2)
    if (!(r2 < D * D) || r2 == 0.0) return;                         // not in contact / coincident (A3)
    const double r = sqrt(r2);
    const double rinv = 1.0 / r;
    const double rdot = (dx * ((double)vj.x - (double)vi.x) + dy * ((double)vj.y - (double)vi.y)
                       + dz * ((double)vj.z - (double)vi.z)) * rinv;
    const double g = (rdot < -(double)a.v_dead) ? (double)a.gamma : (double)a.gamma_beta;  // Eq. 5 : Eq. 6 (A5)
    const double kPi = 3.14159265358979323846;
    double piV;
    if (a.lens_mode == 0) {
        const double h = D - r;
        piV = (kPi / 12.0) * h * h * (2.0 * D + r);
    } else {
        const double R = 0.5 * D;
        piV = kPi * ((4.0 / 3.0) * R * R * R - R * R * r + r * r / 12.0);
    }
    const double c = -g * piV / (double)vi.w * rinv;                // vi.w = m_i
    ax += c * dx; ay += c * dy; az += c * dz;
}

// One contact pair, Eqs. 5/6, as the acceleration it gives element i (x m_i: the caller
// multiplies by 1/m_i).  Same decisions and the same exact fp64 differences as contact_term(); 1/r comes from
// the fp32 MUFU.RSQ seed refined by two Newton steps in fp64 (relative error ~2^-52) instead of a
// double-precision square root and division (~10 instead of ~60 fp64-pipe instructions).
__device__ __forceinline__ void contact_pair(const ContactArgs& a, const float4 pi, const float4 vi, const float4 pj,
                                             const float4 vj, double& fx, double& fy, double& fz)
{
    fx = fy = fz = 0.0;
    const double dx = (double)pj.x - (double)pi.x, dy = (double)pj.y - (double)pi.y, dz = (double)pj.z - (double)pi.z;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double D = (double)pi.w + (double)pj.w;                   // R_i + R_j = 2 R_ij (A2)
    if (!(r2 < D * D) || r2 == 0.0) return;                         // not in contact / coincident (A3)
    double y;
    if (r2 > 1.0e-30) {
        y = (double)rsqrt_approx((float)r2);
        y = y * (1.5 - 0.5 * r2 * y * y);
        y = y * (1.5 - 0.5 * r2 * y * y);
    } else {
        y = 1.0 / sqrt(r2);
    }
    const double r = r2 * y;
    const double rdot = (dx * ((double)vj.x - (double)vi.x) + dy * ((double)vj.y - (double)vi.y)
                       + dz * ((double)vj.z - (double)vi.z)) * y;
    const double g = (rdot < -(double)a.v_dead) ? (double)a.gamma : (double)a.gamma_beta;  // Eq. 5 : Eq. 6 (A5)
    const double kPi = 3.14159265358979323846;
    double piV;
    if (a.lens_mode == 0) {
        const double h = D - r;
        piV = (kPi / 12.0) * h * h * (2.0 * D + r);
    } else {
        const double R = 0.5 * D;
        piV = kPi * ((4.0 / 3.0) * R * R * R - R * R * r + r * r / 12.0);
    }
    const double c = -g * piV * y;
    fx = c * dx; fy = c * dy; fz = c * dz;
}

// Repulsion potential of one contact pair, reading A12: U_rep(r) = int_r^{2R} gamma pi V dr' = gamma pi h^3 (8R - h) / 48
// with h = 2R - r, 2R = R_i + R_j (factored: no cancellation); 0 if the pair is not in contact.  fp64, as contact_pair().
__device__ __forceinline__ double contact_potential(const ContactArgs& a, const float4 pi, const float4 pj)
{
    const double dx = (double)pj.x - (double)pi.x, dy = (double)pj.y - (double)pi.y, dz = (double)pj.z - (double)pi.z;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double D = (double)pi.w + (double)pj.w;
    if (!(r2 < D * D)) return 0.0;                                   // r = 0 (two elements at one point) is a pair like any other here: U_rep(0) = gamma pi R^4, A3
    const double h = D - sqrt(r2);
    return (double)a.gamma * (3.14159265358979323846 / 48.0) * h * h * h * (4.0 * D - h);
}

// Squared gap between a point and an axis-aligned box (0 inside).
__device__ __forceinline__ float point_gap2(const float4 p, const float4 lo, const float4 hi) {
    const float gx = fmaxf(0.f, fmaxf(lo.x - p.x, p.x - hi.x));
    const float gy = fmaxf(0.f, fmaxf(lo.y - p.y, p.y - hi.y));
    const float gz = fmaxf(0.f, fmaxf(lo.z - p.z, p.z - hi.z));
    return gx * gx + gy * gy + gz * gz;
}

constexpr int kCandCap = 128;         // candidate groups buffered per warp before they are processed
constexpr int kHitCap = 40;           // per-lane queue of pairs that passed the fp32 pre-test (a group adds <= 32)
constexpr int kHitFlush = 8;          // the queues are drained once any lane holds this many

// Drain the warp's hit queues: every lane evaluates ITS OWN queued pairs in the order it found them
// (so the fp64 sums have the same fixed order as an immediate evaluation would give), all lanes in
// step -- the fp64 contact term is ~80 instructions, and evaluated at the point of discovery it ran
// with one or two lanes active.
__device__ __forceinline__ void contact_drain(const ContactArgs& a, const uint32_t* __restrict__ hq, int& nh,
                                              const float4 pi, const float4 vi, int lane,
                                              double& ax, double& ay, double& az)
{
    const int mx = __reduce_max_sync(0xffffffffu, nh);
    for (int k = 0; k < mx; ++k) {
        if (k < nh) {
            const int j = (int)hq[k * 32 + lane];
            contact_term(a, pi, vi, a.ps[j], a.vs[j], ax, ay, az);
        }
    }
    nh = 0;
}

// Test the lane's element i against the `cnt` candidate groups listed in cand[]:
// a group is skipped unless some lane's point is within reach of its box; its 32 elements are
// staged in the warp's shared-memory slot (coalesced load, broadcast reads); pairs that pass the
// fp32 pre-test go to the lane's hit queue.
__device__ __forceinline__ void contact_candidates(const ContactArgs& a, const int* __restrict__ cand, int cnt,
                                                   float4* __restrict__ stage, uint32_t* __restrict__ hq, int& nh,
                                                   const float4 pi, const float4 vi,
                                                   bool valid, int lane, double& ax, double& ay, double& az)
{
    const float kSlack = 1.0f + 1.0e-5f;
    for (int q = 0; q < cnt; ++q) {
        const int jg = cand[q];
        const float4 lo = a.gbox[2 * jg], hi = a.gbox[2 * jg + 1];
        const float Db = pi.w + lo.w;
        if (!__any_sync(0xffffffffu, valid && point_gap2(pi, lo, hi) <= Db * Db * kSlack)) continue;
        const int j0 = jg * kGroup;
        const int jn = min(kGroup, a.n - j0);
        // stage the group as four arrays of 32 floats (x, y, z, R; the ragged end far away), so that one
        // broadcast LDS.64 gives a packed pair of elements j and the pre-test runs on FADD2/FFMA2/FMUL2:
        // the same operations in the same order per element as the scalar form, two elements at a time
        float* __restrict__ sx = reinterpret_cast<float*>(stage);
        __syncwarp();
        {
            float4 p = make_float4(kFarAway, kFarAway, kFarAway, 0.f);
            if (lane < jn) p = a.ps[j0 + lane];
            sx[lane] = p.x; sx[32 + lane] = p.y; sx[64 + lane] = p.z; sx[96 + lane] = p.w;
        }
        __syncwarp();
        const f32x2 nx = pk2(-pi.x, -pi.x), ny = pk2(-pi.y, -pi.y), nz = pk2(-pi.z, -pi.z), Ri = pk2(pi.w, pi.w);
        const f32x2 slack2 = pk2(kSlack, kSlack);
#pragma unroll 4
        for (int t = 0; t < kGroup; t += 2) {
            const f32x2 dx = add2(*reinterpret_cast<const f32x2*>(sx + t), nx);
            const f32x2 dy = add2(*reinterpret_cast<const f32x2*>(sx + 32 + t), ny);
            const f32x2 dz = add2(*reinterpret_cast<const f32x2*>(sx + 64 + t), nz);
            const f32x2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
            const f32x2 D = add2(Ri, *reinterpret_cast<const f32x2*>(sx + 96 + t));
            const f32x2 thr = mul2(mul2(D, D), slack2);
            float r0, r1, t0, t1;
            unpk2(r2, r0, r1); unpk2(thr, t0, t1);
            if (r0 <= t0 && valid) { hq[nh * 32 + lane] = (uint32_t)(j0 + t); ++nh; }
            if (r1 <= t1 && valid) { hq[nh * 32 + lane] = (uint32_t)(j0 + t + 1); ++nh; }
        }
        if (__any_sync(0xffffffffu, nh >= kHitFlush)) contact_drain(a, hq, nh, pi, vi, lane, ax, ay, az);
    }
}

// Small n (groups in index order, no sort: every group is a candidate of every other): the
// search above would leave n/32 warps walking all n elements one after the other.  Here a warp
// owns (group of 32 elements i, chunk of `cg` candidate groups) and writes its own slab
// out[chunk][i]; the update kernel adds the slabs in chunk order.
// The work of warp `wid` of that grid; cand [kCandCap], stage [kGroup], hq [kHitCap * 32]: the warp's shared memory.
__device__ __forceinline__ void contact_chunk_warp(const ContactArgs& a, const int cg, const int nchunks, const int wid,
                                                   int* __restrict__ cand, float4* __restrict__ stage,
                                                   uint32_t* __restrict__ hq)
{
    const int lane = threadIdx.x & 31;
    int nh = 0;
    const int ig = wid / nchunks, ch = wid - ig * nchunks;
    if (ig >= a.ngroups) return;
    const int k = ig * kGroup + lane;
    const bool valid = k < a.n;
    const float4 pi = valid ? a.ps[k] : make_float4(kFarAway, kFarAway, kFarAway, 0.f);
    const float4 vi = valid ? a.vs[k] : make_float4(0.f, 0.f, 0.f, 1.f);
    const int g0 = ch * cg, g1 = min(g0 + cg, a.ngroups);
    double ax = 0.0, ay = 0.0, az = 0.0;
    for (int gb = g0; gb < g1; gb += kCandCap) {
        const int cnt = min(kCandCap, g1 - gb);
        __syncwarp();
        for (int q = lane; q < cnt; q += 32) cand[q] = gb + q;
        __syncwarp();
        contact_candidates(a, cand, cnt, stage, hq, nh, pi, vi, valid, lane, ax, ay, az);
    }
    contact_drain(a, hq, nh, pi, vi, lane, ax, ay, az);
    if (valid) a.out[(size_t)ch * a.n + k] = make_float4((float)ax, (float)ay, (float)az, 0.f);
}

__global__ void __launch_bounds__(kThreads)
nb_contact_chunk_kernel(const __grid_constant__ ContactArgs a, const int cg, const int nchunks)
{
    __shared__ int cand_s[kThreads / 32][kCandCap];
    __shared__ float4 stage_s[kThreads / 32][kGroup];
    __shared__ uint32_t hit_s[kThreads / 32][kHitCap * 32];
    const int wib = threadIdx.x >> 5;
    contact_chunk_warp(a, cg, nchunks, (blockIdx.x * kThreads + threadIdx.x) >> 5, cand_s[wib], stage_s[wib], hit_s[wib]);
}

// ---------------------------------------------------------------------------
// Split-j reduction fused with the leapfrog update (rows a4 + a6 + a5).
//   a_i = sum_p src[p][i]  (fixed order, fp64)
//   if acc_out: acc_out[i] = a_i
//   v_i += kick_h * a_i ;  x_i += drift_dt * v_i        (either may be 0)
//   if advance: step += 1, R_s = ramp(step)             (expanding-star rule)
struct UpdateArgs {
    const double* acc64;               // chain mode: [6][n] fp64 sums (a_i side x,y,z; reaction x,y,z), else nullptr
    const float4* src;                 // [nsrc][n]
    float4* acc_out;                   // may be null; may alias src when nsrc == 1
    float4* posm;
    float4* vel;
    DevState* dev;
    int n, nsrc;
    float kick_h, drift_dt;
    float vscale;                      // relaxation (f2): v <- vscale (v + kick_h a); 1 for the plain leapfrog
    int advance;
};

// Expanding-star rule (A8): step count n and R_s(n), linear in n over n_ramp steps, evaluated
// in fp64 with explicit roundings (no contraction) and rounded once to the fp32 model parameter.
__device__ __forceinline__ float ramp_radius(double R_start, double R_end, long long n_ramp, long long nstep)
{
    double Rs = R_start;
    if (n_ramp > 0) {
        const long long nn = nstep < n_ramp ? nstep : n_ramp;
        Rs = __dadd_rn(R_start, __ddiv_rn(__dmul_rn(__dsub_rn(R_end, R_start), (double)nn), (double)n_ramp));
    }
    return (float)Rs;
}

__device__ __forceinline__ void set_step(DevState* d, long long nstep)
{
    d->step = nstep;
    for (int s = 0; s < 2; ++s) d->R[s] = ramp_radius(d->R_start[s], d->R_end[s], d->n_ramp, nstep);
}

// Element i of the update, given a_i: kick, drift (new position and velocity through p, v: valid if moved).
__device__ __forceinline__ void apply_update(const UpdateArgs& u, const int i, const float ax, const float ay, const float az,
                                             float4& p, float4& v)
{
    if (u.acc_out) u.acc_out[i] = make_float4(ax, ay, az, 0.f);
    if (u.kick_h != 0.f || u.drift_dt != 0.f || u.vscale != 1.f) {
        v = u.vel[i];
        v.x = fmaf(u.kick_h, ax, v.x);
        v.y = fmaf(u.kick_h, ay, v.y);
        v.z = fmaf(u.kick_h, az, v.z);
        if (u.vscale != 1.f) { v.x *= u.vscale; v.y *= u.vscale; v.z *= u.vscale; }
        u.vel[i] = v;
        if (u.drift_dt != 0.f) {
            p = u.posm[i];
            p.x = fmaf(u.drift_dt, v.x, p.x);
            p.y = fmaf(u.drift_dt, v.y, p.y);
            p.z = fmaf(u.drift_dt, v.z, p.z);
            u.posm[i] = p;
        }
    }
}

// Element i of the update: a_i = sum of the slabs in slab order (fp64), then kick and drift.  Returns a_i.
__device__ __forceinline__ float4 update_element(const UpdateArgs& u, const int i, float4& p, float4& v)
{
    double sx = 0.0, sy = 0.0, sz = 0.0;
    if (u.acc64) {
        const size_t n = (size_t)u.n;
        const double* q = u.acc64 + i;
        sx = q[0] + q[3 * n]; sy = q[n] + q[4 * n]; sz = q[2 * n] + q[5 * n];
    }
#pragma unroll 8
    for (int q = 0; q < u.nsrc; ++q) {
        const float4 t = u.src[(size_t)q * u.n + i];
        sx += (double)t.x; sy += (double)t.y; sz += (double)t.z;
    }
    const float ax = (float)sx, ay = (float)sy, az = (float)sz;
    apply_update(u, i, ax, ay, az, p, v);
    return make_float4(ax, ay, az, 0.f);
}

__global__ void __launch_bounds__(256)
nb_reduce_update_kernel(const __grid_constant__ UpdateArgs u)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < u.n) {
        float4 p, v;
        update_element(u, i, p, v);
    }
    if (u.advance && blockIdx.x == 0 && threadIdx.x == 0) set_step(u.dev, u.dev->step + 1);
}

// nb_set_step(): restore the step count of a checkpointed run; the radii follow from it.
__global__ void nb_set_step_kernel(DevState* dev, long long step) { set_step(dev, step); }

// star[] must be 0...0 1...1; counts the zeros into dev->n1, flags violations.
__global__ void nb_validate_star_kernel(const int32_t* __restrict__ star, int n, DevState* dev)
{
    int zeros = 0, bad = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int s = star[i];
        if (s != 0 && s != 1) bad = 1;
        if (i + 1 < n && star[i + 1] < s) bad = 1;
        zeros += (s == 0);
    }
    if (zeros) atomicAdd(&dev->n1, zeros);
    if (bad) atomicOr(&dev->bad, 1);
}

// ---------------------------------------------------------------------------
// Diagnostics (row a7).  Block-level fp64 partials, summed on the host in fixed order.
constexpr int kMomentCols = 10;   // KE, Px,Py,Pz, Lx,Ly,Lz, Fx,Fy,Fz

__device__ __forceinline__ double block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int k = 0; k < (int)(blockDim.x >> 5); ++k) r += sh[k];
    return r;   // valid in thread 0
}

__global__ void __launch_bounds__(256)
nb_moments_kernel(const float4* __restrict__ posm, const float4* __restrict__ vel,
                  const float4* __restrict__ acc, int n, double* __restrict__ out /*[grid][10]*/)
{
    __shared__ double sh[8];
    double q[kMomentCols];
    for (int c = 0; c < kMomentCols; ++c) q[c] = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 p = posm[i], v = vel[i], a = acc[i];
        const double m = p.w, x = p.x, y = p.y, z = p.z, vx = v.x, vy = v.y, vz = v.z;
        q[0] += 0.5 * m * (vx * vx + vy * vy + vz * vz);
        q[1] += m * vx; q[2] += m * vy; q[3] += m * vz;
        q[4] += m * (y * vz - z * vy);
        q[5] += m * (z * vx - x * vz);
        q[6] += m * (x * vy - y * vx);
        q[7] += m * (double)a.x; q[8] += m * (double)a.y; q[9] += m * (double)a.z;
    }
    for (int c = 0; c < kMomentCols; ++c) {
        const double r = block_sum(q[c], sh);
        if (threadIdx.x == 0) out[(size_t)blockIdx.x * kMomentCols + c] = r;
    }
}

// Potential energies: per block, sum_i m_i * sum_{j > i} G m_j/(r+eps)  and
// sum_i sum_{j > i, contact} U_rep(r; R_ij)   (each unordered pair counted once: thread i walks only
// the tiles from its own on; the blocks are launched in index order, longest first).
struct PotArgs {
    const float4* __restrict__ posm;
    const DevState* __restrict__ dev;
    double* __restrict__ out;          // [grid][2]
    int n, n1;
    float G, eps, gamma;
};

__global__ void __launch_bounds__(kThreads)
nb_potential_kernel(const __grid_constant__ PotArgs a)
{
    constexpr int TJ = 256;
    __shared__ float4 sj[TJ];
    __shared__ double sh[8];
    const int tid = threadIdx.x;
    const int i = blockIdx.x * kThreads + tid;
    const float R0 = a.dev->R[0], R1 = a.dev->R[1];
    float4 pi = make_float4(-kFarAway, -kFarAway, -kFarAway, 0.f);
    if (i < a.n) pi = a.posm[i];
    const float Ri = star_radius(min(i, a.n - 1), a.n1, R0, R1);
    const float Dmax = Ri + fmaxf(R0, R1);
    const float kPi = 3.14159265358979f;
    double phi = 0.0, urep = 0.0;
    const int njt = (a.n + TJ - 1) / TJ;
    for (int t = (blockIdx.x * kThreads) / TJ; t < njt; ++t) {    // only the tiles that hold some j > i
        __syncthreads();
        for (int l = tid; l < TJ; l += kThreads) {
            const int j = t * TJ + l;
            sj[l] = j < a.n ? a.posm[j] : make_float4(kFarAway, kFarAway, kFarAway, 0.f);
        }
        __syncthreads();
        float ph = 0.f;
#pragma unroll 4
        for (int jj = 0; jj < TJ; ++jj) {
            const float4 pj = sj[jj];
            const int j = t * TJ + jj;
            const float dx = pj.x - pi.x, dy = pj.y - pi.y, dz = pj.z - pi.z;
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, kTinyR2)));
            const float r = r2 * rsqrt_approx(r2);
            const float w = (j > i) ? pj.w : 0.f;                    // every unordered pair once
            ph = fmaf(w, rcp_approx(r + a.eps), ph);
            if (a.gamma > 0.f && r2 < Dmax * Dmax && j > i && j < a.n) {
                const float D = Ri + star_radius(j, a.n1, R0, R1);
                const float rr = sqrtf(r2);
                if (rr < D) {
                    // A12 in factored form: with h = 2R - r,  U_rep = gamma pi h^3 (8R - h)/48
                    // (= gamma pi (R^4 - 4/3 R^3 r + 1/2 R^2 r^2 - r^4/48), no cancellation)
                    const float h = D - rr;
                    urep += (double)(a.gamma * (kPi / 48.0f) * h * h * h * (4.0f * D - h));
                }
            }
        }
        phi += (double)ph;
    }
    const double e1 = block_sum((double)a.G * (double)pi.w * phi, sh);
    const double e2 = block_sum(i < a.n ? urep : 0.0, sh);
    if (tid == 0) { a.out[2 * (size_t)blockIdx.x] = e1; a.out[2 * (size_t)blockIdx.x + 1] = e2; }
}

// Row a7 for n >= 8,192: U_grav = -sum_{i<j} G m_i m_j / (r + eps) over pairs of super-tiles (A <= B), one CTA each,
// in the packed form of the symmetric gravity kernel: B staged in shared memory as packed pairs (broadcast LDS.64),
// NI elements i of A per lane, per pair one MUFU.RSQ (y = 1/r, r = r^2 y) and
//   near pairs of super-tiles: one MUFU.RCP, 1/(r + eps) -- the XU pipe bounds them at the N^2 MUFU of a force evaluation;
//   FAR pairs (bounding boxes at least 100 eps apart, so u = eps/r <= 0.01): no second MUFU, the factor 1/(1 + u) as
//   1 - u + u^2 - u^3 (truncation error u^4 <= 1e-8 relative), i.e. y (1 + y (-eps + y (eps^2 - eps^3 y))): three FFMA2 and
//   one FMUL2 instead -- the FMA pipe bounds them, at 22 instead of 32 cycles per packed evaluation.
// The elements are taken in the cell-list order of the contact pass when there is one (nb_energy runs it first, in
// energy mode): super-tiles are then thin pencils of cells and ~90 % of the same-star pairs are far as well; in the
// caller's order only the pairs of super-tiles from different stars are.  Either way the sum is over the same pairs.
// fp32 terms in chains of <= 128, flushed into fp64; one fp64 partial per CTA, summed on the host in CTA order.  A
// diagonal CTA (A == B) counts every ordered pair but the self pair (masked by index) and halves the sum.
// U_rep comes from the cell list (nb_cells.cuh, energy mode).
struct PotPairArgs {
    const float4* __restrict__ px;     // [n] x,y,z,.   (posm, or the sorted copy ps)
    const float4* __restrict__ pm;     // [n] .,.,.,m   (posm, or the sorted copy vs)
    const float4* __restrict__ box;    // [T][2] bounding box of every super-tile (lo, hi)
    double* __restrict__ out;          // [T (T + 1) / 2]
    int n, T;
    float G, eps;
};

// Bounding boxes of the super-tiles of S elements: one block per super-tile.
__global__ void __launch_bounds__(256)
nb_tile_bbox_kernel(const float4* __restrict__ px, int n, int S, float4* __restrict__ box)
{
    __shared__ float sh[6][8];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
    const long long e0 = (long long)blockIdx.x * S;
    for (int k = threadIdx.x; k < S && e0 + k < n; k += 256) {
        const float4 q = px[e0 + k];
        lo[0] = fminf(lo[0], q.x); lo[1] = fminf(lo[1], q.y); lo[2] = fminf(lo[2], q.z);
        hi[0] = fmaxf(hi[0], q.x); hi[1] = fmaxf(hi[1], q.y); hi[2] = fmaxf(hi[2], q.z);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float a = warp_min(lo[c]), b = warp_max(hi[c]);
        if (l == 0) { sh[c][w] = a; sh[3 + c][w] = b; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        float q[6];
        for (int c = 0; c < 3; ++c) {
            q[c] = sh[c][0]; q[3 + c] = sh[3 + c][0];
            for (int k = 1; k < 8; ++k) { q[c] = fminf(q[c], sh[c][k]); q[3 + c] = fmaxf(q[3 + c], sh[3 + c][k]); }
        }
        box[2 * blockIdx.x] = make_float4(q[0], q[1], q[2], 0.f);
        box[2 * blockIdx.x + 1] = make_float4(q[3], q[4], q[5], 0.f);
    }
}

constexpr float kPotFarGap = 100.f;    // a pair of super-tiles is FAR if its boxes are at least this many eps apart

template <int NI, bool DIAG, bool FAR>
__device__ __forceinline__ void pot_step(const f32x2 X, const f32x2 Y, const f32x2 Z, const f32x2 M, const int j0,
                                         const float (&nxi)[NI], const float (&nyi)[NI], const float (&nzi)[NI],
                                         const int (&ei)[NI], const f32x2 eps2, const f32x2 neps, const f32x2 e2,
                                         const f32x2 ne3, f32x2 (&acc)[NI])
{
    const f32x2 tiny2 = pk2(kTinyR2, kTinyR2);
    f32x2 r2[NI], y[NI];
#pragma unroll
    for (int i = 0; i < NI; ++i) {
        const f32x2 dx = add2(X, pk2(nxi[i], nxi[i])), dy = add2(Y, pk2(nyi[i], nyi[i])), dz = add2(Z, pk2(nzi[i], nzi[i]));
        r2[i] = fma2(dx, dx, tiny2); r2[i] = fma2(dy, dy, r2[i]); r2[i] = fma2(dz, dz, r2[i]);
    }
#pragma unroll
    for (int i = 0; i < NI; ++i) {
        float a0, b0;
        unpk2(r2[i], a0, b0);
        y[i] = pk2(rsqrt_approx(a0), rsqrt_approx(b0));
    }
    if constexpr (FAR) {                             // 1/(r + eps) = y / (1 + eps y) = y (1 + y (-eps + y (eps^2 - eps^3 y)))
        const f32x2 one = pk2(1.f, 1.f);
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            f32x2 q = fma2(y[i], ne3, e2);
            q = fma2(y[i], q, neps);
            q = fma2(y[i], q, one);
            acc[i] = fma2(M, mul2(y[i], q), acc[i]);                                  // m_j / (r + eps)
        }
    } else {
        f32x2 sm[NI];
#pragma unroll
        for (int i = 0; i < NI; ++i) sm[i] = fma2(r2[i], y[i], eps2);             // r + eps
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            float a0, b0;
            unpk2(sm[i], a0, b0);
            f32x2 w = M;
            if (DIAG) {                              // the self pair does not count
                float m0, m1;
                unpk2(M, m0, m1);
                w = pk2(j0 == ei[i] ? 0.f : m0, j0 + 1 == ei[i] ? 0.f : m1);
            }
            acc[i] = fma2(w, pk2(rcp_approx(a0), rcp_approx(b0)), acc[i]);        // m_j / (r + eps)
        }
    }
}

// MODE 0: off-diagonal pair of super-tiles, near; 1: diagonal; 2: off-diagonal, far.
template <int S, int NI, int NT, int MODE>
__device__ __forceinline__ double pot_sweep(const PotPairArgs& a, const int A, const int B,
                                            const float2* __restrict__ X2, const float2* __restrict__ Y2,
                                            const float2* __restrict__ Z2, const float2* __restrict__ M2)
{
    constexpr int IPR = NT * NI;                     // elements i per round
    const int tid = threadIdx.x;
    const f32x2 eps2 = pk2(a.eps, a.eps), neps = pk2(-a.eps, -a.eps), e2 = pk2(a.eps * a.eps, a.eps * a.eps),
                ne3 = pk2(-a.eps * a.eps * a.eps, -a.eps * a.eps * a.eps);
    double total = 0.0;
#pragma unroll 1
    for (int r = 0; r < S / IPR; ++r) {
        float nxi[NI], nyi[NI], nzi[NI], mi[NI];
        int ei[NI];
        double phi[NI];
#pragma unroll
        for (int i = 0; i < NI; ++i) {
            ei[i] = A * S + r * IPR + i * NT + tid;
            float4 q = make_float4(-kFarAway, -kFarAway, -kFarAway, 0.f);
            if (ei[i] < a.n) { q = a.px[ei[i]]; q.w = a.pm[ei[i]].w; }
            nxi[i] = -q.x; nyi[i] = -q.y; nzi[i] = -q.z; mi[i] = q.w;
            phi[i] = 0.0;
        }
#pragma unroll 1
        for (int p0 = 0; p0 < S / 2; p0 += 64) {
            f32x2 acc[NI];
#pragma unroll
            for (int i = 0; i < NI; ++i) acc[i] = pk2(0.f, 0.f);
#pragma unroll 4
            for (int p = p0; p < p0 + 64; ++p) {
                const f32x2 X = *reinterpret_cast<const f32x2*>(X2 + p), Y = *reinterpret_cast<const f32x2*>(Y2 + p),
                            Z = *reinterpret_cast<const f32x2*>(Z2 + p), M = *reinterpret_cast<const f32x2*>(M2 + p);
                pot_step<NI, MODE == 1, MODE == 2>(X, Y, Z, M, B * S + 2 * p, nxi, nyi, nzi, ei, eps2, neps, e2, ne3, acc);
            }
#pragma unroll
            for (int i = 0; i < NI; ++i) {
                float l, h;
                unpk2(acc[i], l, h);
                phi[i] += (double)l + (double)h;
            }
        }
#pragma unroll
        for (int i = 0; i < NI; ++i) total += (double)mi[i] * phi[i];
    }
    return total;
}

template <int S, int NI, int NT>
__global__ void __launch_bounds__(NT, 3)
nb_pot_pair_kernel(const __grid_constant__ PotPairArgs a)
{
    extern __shared__ float4 pot_smem[];             // X2, Y2, Z2, M2: 4 arrays of S/2 float2 = 16 S bytes
    __shared__ double sh[NT / 32];
    float2* __restrict__ X2 = reinterpret_cast<float2*>(pot_smem);
    float2* __restrict__ Y2 = X2 + S / 2;
    float2* __restrict__ Z2 = Y2 + S / 2;
    float2* __restrict__ M2 = Z2 + S / 2;
    static_assert(S % (NT * NI) == 0 && (S / 2) % 64 == 0, "whole rounds; whole flush intervals");
    const int tid = threadIdx.x;
    int A, B;
    {
        const long long T = a.T, Mo = T * (T - 1) / 2, b = blockIdx.x;
        if (b >= Mo) { A = B = (int)(b - Mo); }
        else {
            const double t2 = 2.0 * (double)T - 1.0;
            long long r = (long long)((t2 - sqrt(t2 * t2 - 8.0 * (double)b)) * 0.5);
            if (r < 0) r = 0;
            while (r > 0 && r * (2 * T - r - 1) / 2 > b) --r;
            while ((r + 1) * (2 * T - r - 2) / 2 <= b) ++r;
            A = (int)r;
            B = (int)(b - r * (2 * T - r - 1) / 2 + r + 1);
        }
    }
    for (int p = tid; p < S / 2; p += NT) {          // pair p holds elements 2 p and 2 p + 1 of B
        const int e0 = B * S + 2 * p, e1 = e0 + 1;
        float4 q0 = make_float4(kFarAway, kFarAway, kFarAway, 0.f), q1 = q0;
        if (e0 < a.n) { q0 = a.px[e0]; q0.w = a.pm[e0].w; }
        if (e1 < a.n) { q1 = a.px[e1]; q1.w = a.pm[e1].w; }
        X2[p] = make_float2(q0.x, q1.x); Y2[p] = make_float2(q0.y, q1.y); Z2[p] = make_float2(q0.z, q1.z);
        M2[p] = make_float2(q0.w, q1.w);
    }
    __syncthreads();
    // far: every r of the pair of super-tiles is at least kPotFarGap eps (and more than nothing)
    const float gap2 = box_gap2(a.box[2 * A], a.box[2 * A + 1], a.box[2 * B], a.box[2 * B + 1]);
    const float need = kPotFarGap * a.eps;
    const bool far = A != B && gap2 > 0.f && gap2 >= need * need;
    double total;
    if (A == B)   total = 0.5 * pot_sweep<S, NI, NT, 1>(a, A, B, X2, Y2, Z2, M2);
    else if (far) total = pot_sweep<S, NI, NT, 2>(a, A, B, X2, Y2, Z2, M2);
    else          total = pot_sweep<S, NI, NT, 0>(a, A, B, X2, Y2, Z2, M2);
    total *= (double)a.G;
    const double rsum = block_sum(total, sh);
    if (tid == 0) a.out[blockIdx.x] = rsum;
}

// ---------------------------------------------------------------------------
// Row f3: mass transfer through L1 (A18).
// Pass 1: per star (by membership: star 0 = indices < n1) M, sum m x, sum m v -- block partials.
constexpr int kXferCols1 = 14;        // per star: M, Mx, My, Mz, Mvx, Mvy, Mvz
constexpr int kXferCols2 = 12;        // Mcross[2], Min[2], Mout[2], Ldisk[2][3]

__global__ void __launch_bounds__(256)
nb_star_moments_kernel(const float4* __restrict__ posm, const float4* __restrict__ vel, int n, int n1,
                       double* __restrict__ out /*[grid][14]*/)
{
    __shared__ double sh[8];
    double q[kXferCols1];
    for (int c = 0; c < kXferCols1; ++c) q[c] = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 p = posm[i], v = vel[i];
        const double m = p.w;
        double* t = q + (i < n1 ? 0 : 7);
        t[0] += m;
        t[1] += m * (double)p.x; t[2] += m * (double)p.y; t[3] += m * (double)p.z;
        t[4] += m * (double)v.x; t[5] += m * (double)v.y; t[6] += m * (double)v.z;
    }
    for (int c = 0; c < kXferCols1; ++c) {
        const double r = block_sum(q[c], sh);
        if (threadIdx.x == 0) out[(size_t)blockIdx.x * kXferCols1 + c] = r;
    }
}

// Between the passes, on the device (so a record per step needs no host round trip): star centres and masses from
// pass 1's block partials (summed in block order), the L1 plane by the force balance along the line of centres
// (Newton iteration, as nb_l1_distance() on the host), the lobe radii by Eq. 3.
struct XferGeom {
    double X[2][3], V[2][3], e[3], d0, rL[2], a, M[2];
    double* out;                       // the 32-double record this evaluation writes (null: dropped)
    long long step;
    int valid;                         // both stars present and apart: pass 2 has something to decide
};

__device__ inline double dev_l1_distance(double q)            // distance of L1 from the primary, separation 1, q = m2/m1 <= 1
{
    const double mu2 = q / (1.0 + q), mu1 = 1.0 - mu2;
    double s = 1.0 - cbrt(mu2 / 3.0);
    for (int it = 0; it < 100; ++it) {
        const double t = 1.0 - s;
        const double f = -mu1 / (s * s) + mu2 / (t * t) + (s - mu2);
        const double df = 2.0 * mu1 / (s * s * s) + 2.0 * mu2 / (t * t * t) + 1.0;
        const double sn = s - f / df;
        if (!(sn > 0.0 && sn < 1.0)) { s = 0.5 * (s + (sn <= 0.0 ? 0.0 : 1.0)); continue; }
        if (fabs(sn - s) < 1e-15) { s = sn; break; }
        s = sn;
    }
    return s;
}

__device__ inline double dev_roche_lobe_radius(double mass_ratio, double k)
{
    const double c = cbrt(mass_ratio);
    return 0.49 * c * c / (k * c * c + log1p(c));                // Eq. 3
}

// rows < 0: the record goes to series[0..31]; else to row `step count` of series[rows][32], dropped when the run is past it.
__global__ void __launch_bounds__(32)
nb_transfer_geometry_kernel(const double* __restrict__ part1 /*[blocks][14]*/, int blocks, double k_lobe,
                            const DevState* __restrict__ dev, double* series, long long rows, XferGeom* __restrict__ g)
{
    __shared__ double q[kXferCols1];
    const int t = threadIdx.x;
    if (t < kXferCols1) {
        double sum = 0.0;
        for (int b = 0; b < blocks; ++b) sum += part1[(size_t)b * kXferCols1 + t];
        q[t] = sum;
    }
    __syncthreads();
    if (t != 0) return;
    const long long step = dev->step;
    double* out = rows < 0 ? series : (step < rows ? series + 32 * step : nullptr);
    g->out = out; g->step = step; g->valid = 0;
    const double M0 = q[0], M1 = q[7];
    g->M[0] = M0; g->M[1] = M1;
    for (int s = 0; s < 2; ++s) {
        const double M = s ? M1 : M0;
        for (int k = 0; k < 3; ++k) {
            g->X[s][k] = M > 0.0 ? q[7 * s + 1 + k] / M : 0.0;
            g->V[s][k] = M > 0.0 ? q[7 * s + 4 + k] / M : 0.0;
        }
    }
    g->a = 0.0; g->d0 = 0.0; g->rL[0] = g->rL[1] = 0.0; g->e[0] = g->e[1] = g->e[2] = 0.0;
    if (!(M0 > 0.0 && M1 > 0.0)) return;                         // one star only: nothing to transfer
    double d[3], a2 = 0.0;
    for (int k = 0; k < 3; ++k) { d[k] = g->X[1][k] - g->X[0][k]; a2 += d[k] * d[k]; }
    const double a = sqrt(a2);
    if (!(a > 0.0)) return;
    for (int k = 0; k < 3; ++k) g->e[k] = d[k] / a;
    g->a = a;
    // L1 along the line of centres, measured from star 0 (dev_l1_distance is measured from the primary)
    g->d0 = M1 <= M0 ? a * dev_l1_distance(M1 / M0) : a * (1.0 - dev_l1_distance(M0 / M1));
    g->rL[0] = a * dev_roche_lobe_radius(M0 / M1, k_lobe);       // Eq. 3: the star's own mass in the numerator
    g->rL[1] = a * dev_roche_lobe_radius(M1 / M0, k_lobe);
    g->valid = 1;
}

// Pass 2: every decision in fp64 on the fp32 coordinates.
struct XferArgs {
    const float4* __restrict__ posm;
    const float4* __restrict__ vel;
    const XferGeom* __restrict__ g;
    double* __restrict__ out;          // [grid][12]
    int n, n1;
};

__global__ void __launch_bounds__(256)
nb_transfer_kernel(const __grid_constant__ XferArgs a)
{
    __shared__ double sh[8];
    __shared__ XferGeom g;
    if (threadIdx.x == 0) g = *a.g;
    __syncthreads();
    double q[kXferCols2];
    for (int c = 0; c < kXferCols2; ++c) q[c] = 0.0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; g.valid && i < a.n; i += gridDim.x * blockDim.x) {
        const float4 p = a.posm[i], v = a.vel[i];
        const int s = i < a.n1 ? 0 : 1, o = 1 - s;
        const double m = p.w;
        const double x0 = (double)p.x - g.X[0][0], y0 = (double)p.y - g.X[0][1], z0 = (double)p.z - g.X[0][2];
        const double x1 = (double)p.x - g.X[1][0], y1 = (double)p.y - g.X[1][1], z1 = (double)p.z - g.X[1][2];
        const double u = x0 * g.e[0] + y0 * g.e[1] + z0 * g.e[2];
        const double r0 = sqrt(x0 * x0 + y0 * y0 + z0 * z0), r1 = sqrt(x1 * x1 + y1 * y1 + z1 * z1);
        if (s == 0 ? (u > g.d0) : (u < g.d0)) q[s] += m;                       // beyond the L1 plane
        if ((o == 0 ? r0 : r1) < g.rL[o]) {                                    // inside the other star's lobe sphere
            q[2 + s] += m;
            const double rx = o == 0 ? x0 : x1, ry = o == 0 ? y0 : y1, rz = o == 0 ? z0 : z1;
            const double wx = (double)v.x - g.V[o][0], wy = (double)v.y - g.V[o][1], wz = (double)v.z - g.V[o][2];
            q[6 + 3 * s] += m * (ry * wz - rz * wy);
            q[7 + 3 * s] += m * (rz * wx - rx * wz);
            q[8 + 3 * s] += m * (rx * wy - ry * wx);
        }
        if (r0 > g.rL[0] && r1 > g.rL[1]) q[4 + s] += m;                       // outside both
    }
    for (int c = 0; c < kXferCols2; ++c) {
        const double r = block_sum(q[c], sh);
        if (threadIdx.x == 0) a.out[(size_t)blockIdx.x * kXferCols2 + c] = r;
    }
}

// The record (layout: nb.h, nb_transfer_diagnostics): pass 2's block partials summed in block order.
__global__ void __launch_bounds__(32)
nb_transfer_finish_kernel(const double* __restrict__ part2 /*[blocks][12]*/, int blocks, const XferGeom* __restrict__ g)
{
    double* out = g->out;
    if (!out) return;
    const int t = threadIdx.x;
    double v = 0.0;
    if (t == 0) v = g->M[0];
    else if (t == 1) v = g->M[1];
    else if (t == 2) v = g->a;
    else if (t == 3) v = g->d0;
    else if (t == 4) v = g->rL[0];
    else if (t == 5) v = g->rL[1];
    else if (t < 6 + kXferCols2) { for (int b = 0; b < blocks; ++b) v += part2[(size_t)b * kXferCols2 + (t - 6)]; }
    else if (t < 24) v = g->X[(t - 18) / 3][(t - 18) % 3];
    else if (t < 30) v = g->V[(t - 24) / 3][(t - 24) % 3];
    else if (t == 30) v = (double)g->step;
    out[t] = v;
}

// ---------------------------------------------------------------------------
// Row f4: headless point splat in place of the paper's OpenGL viewer
// (A19).  Orthographic projection on two coordinate axes; the pixel index
// is decided in float32 with one rounding per operation (no FMA contraction), the same
// arithmetic the oracle spells out; counts are integer atomics, so the image is exact.
__global__ void __launch_bounds__(256)
nb_splat_kernel(const float4* __restrict__ posm, int n, int n1, float cu, float cv, float scale,
                int axis_u, int axis_v, int W, int H, unsigned int* __restrict__ image /*[2][H][W]*/)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 p = posm[i];
    const float xu = axis_u == 0 ? p.x : (axis_u == 1 ? p.y : p.z);
    const float xv = axis_v == 0 ? p.x : (axis_v == 1 ? p.y : p.z);
    const float fu = floorf(__fadd_rn(__fmul_rn(__fsub_rn(xu, cu), scale), 0.5f * (float)W));
    const float fv = floorf(__fadd_rn(__fmul_rn(__fsub_rn(xv, cv), scale), 0.5f * (float)H));
    if (!(fu >= 0.f && fu < (float)W && fv >= 0.f && fv < (float)H)) return;
    const int s = i < n1 ? 0 : 1;
    atomicAdd(&image[((size_t)s * H + (int)fv) * W + (int)fu], 1u);
}

}  // namespace nb
