// nb_kernels.cuh -- sm_100a kernels of the all-pairs binary-star element model.
//
// Hot path:
//   a2/a3  nb_force_kernel        all-pairs Eq. 4 gravity with the contact terms of
//                                 Eqs. 5/6 on a warp-voted slow path
//   a4/a6  nb_reduce_update_kernel split-j partial-sum reduction fused with the
//                                 leapfrog kick/drift and the expanding-star rule
//
//   a7     nb_potential_kernel / nb_moments_kernel   diagnostics for nb_energy
//
// The force kernel is bound by the plain FP32 ALUs (FMA pipe, with the XU pipe close
// behind): per interaction 13 FP32 operations issued as packed FFMA2/FADD2/FMUL2,
// one MUFU.RSQ and half a MUFU.RCP.  Not a dense contraction: no tensor cores.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nb {

constexpr int kThreads = 128;          // 4 warps: one per SM sub-partition
constexpr float kTinyR2 = 1.0e-20f;    // added to r^2: keeps the self pair (d = 0) finite, even for eps = 0
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

struct ForceArgs {
    const float4* __restrict__ posm;   // [n] x,y,z,m
    const float4* __restrict__ vel;    // [n] vx,vy,vz,-
    const DevState* __restrict__ dev;
    float4* __restrict__ part;         // [nsplit][n] partial accelerations
    int n, n1, nib, nsplit, njt;
    float G, eps;
    float gamma, gamma_beta;           // Eq. 5 / Eq. 6 strengths
    float v_dead;
    int lens_mode;
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

// Radius of the star an element index belongs to (star 0 first, then star 1).
__device__ __forceinline__ float star_radius(int idx, int n1, float R0, float R1) {
    return idx < n1 ? R0 : R1;
}

// Slow path: the contact term of one (i, j) pair, Eqs. 5/6, added
// to the fp64 accumulators of i: a_i -= g pi V(r; R_ij) / m_i * d/r if r < R_i + R_j.
// d is the fp32 difference the fast path used (exact for near pairs); everything
// else is evaluated in double (B200 has full-rate-class fp64; ~5/N of all pairs come
// here, and h = 2R - r cancels badly in fp32 near first contact).
// lens_mode 0: pi V = pi (D - r)^2 (2D + r) / 12 with D = 2 R_ij (factored displaced
// volume, A1); lens_mode 1: the polynomial as printed, last term r^2/12.
__device__ __forceinline__ void contact_term(const ForceArgs& a, int i, int j, float dxf, float dyf, float dzf,
                                             float R0, float R1, double& ax, double& ay, double& az)
{
    if (i >= a.n || j >= a.n || i == j) return;
    const double dx = dxf, dy = dyf, dz = dzf;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double D = (double)star_radius(i, a.n1, R0, R1) + (double)star_radius(j, a.n1, R0, R1);  // 2 R_ij (A2)
    if (!(r2 < D * D) || r2 == 0.0) return;                // not in contact / coincident (A3)
    const double r = sqrt(r2);
    const double rinv = 1.0 / r;
    const float4 vi = a.vel[i], vj = a.vel[j];
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
    const double c = -g * piV / (double)a.posm[i].w * rinv;
    ax += c * dx; ay += c * dy; az += c * dz;
}

// All-pairs acceleration, one CTA per (i-block, j-split).
//
// Each thread keeps I (even) elements i in registers as I/2 packed pairs; the CTA
// streams its j range through shared memory in tiles of TJ elements
// (double-buffered, one barrier per tile); every LDS.128 of (x_j, y_j, z_j, G m_j)
// is a warp broadcast reused for I pairs.  Per pair of interactions (one packed
// lane pair) the loop issues 13 packed FP32 instructions (FADD2 x3, FFMA2 x7,
// FMUL2 x3), 2 MUFU.RSQ, and ONE MUFU.RCP shared by the two lanes through a
// two-term Montgomery inversion (3 scalar FMUL): 1/t0 = t1/(t0 t1), 1/t1 = t0/(t0 t1),
// with t = (r+eps)^2 >= eps^2 so the product cannot underflow.  That moves the
// bound from the XU pipe (16 lanes/clk/SM) to the FMA pipe.
// Per-tile fp32 partial sums are flushed into fp64 accumulators (short chains).
// Contacts (CONTACT): the minimum r^2 over a group of kGroupJ elements j (FMNMX3 on
// the ALU pipe) is tested once per group against the tile's (R_i+R_j)^2 bound;
// candidate groups go to a small per-thread queue in shared memory and are
// resolved after the tile's loop by contact_term().
constexpr int kQueueDepth = 16;
#ifndef NB_MINB4
#define NB_MINB4 4      // resident CTAs/SM the I=4 kernel is compiled for (register cap 65536/(128*NB_MINB4))
#endif
#ifndef NB_UNROLL
#define NB_UNROLL 4
#endif
constexpr int kGroupJ = NB_UNROLL;    // elements j per unrolled group = granularity of the contact test

template <int I, int TJ, bool CONTACT>
__global__ void __launch_bounds__(kThreads, (I >= 4 ? NB_MINB4 : 6))
nb_force_kernel(const __grid_constant__ ForceArgs a)
{
    static_assert(I % 2 == 0 && TJ % kThreads == 0 && TJ % kGroupJ == 0 && TJ / kGroupJ <= 256,
                  "packed pairs; whole groups; group index fits a byte");
    constexpr int H = I / 2;                        // packed pairs per thread
    constexpr int LPT = TJ / kThreads;              // tile loads per thread
    __shared__ float4 sj[2][TJ];
    __shared__ unsigned char queue[CONTACT ? kQueueDepth * kThreads : 1];

    const int tid = threadIdx.x;
    const int ib = blockIdx.x % a.nib;
    const int sp = blockIdx.x / a.nib;
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

    const float R0 = a.dev->R[0], R1 = a.dev->R[1];
    const int t0 = (int)(((long long)sp * a.njt) / a.nsplit);
    const int t1 = (int)(((long long)(sp + 1) * a.njt) / a.nsplit);

    double accx[I], accy[I], accz[I];
#pragma unroll
    for (int k = 0; k < I; ++k) accx[k] = accy[k] = accz[k] = 0.0;

    // contact bound of this thread's elements: (max R_i + max R_j)^2 per tile
    float Ri_max = 0.f;
    if (CONTACT) {
        const int ilast = min(ibase + (I - 1) * kThreads, a.n - 1);
        Ri_max = (ibase < a.n1 && ilast >= a.n1) ? fmaxf(R0, R1)
                                                 : star_radius(min(ibase, a.n - 1), a.n1, R0, R1);
    }

    float4 pre[LPT];
    auto load_tile = [&](int t) {
#pragma unroll
        for (int l = 0; l < LPT; ++l) {
            const int j = t * TJ + l * kThreads + tid;
            if (j < a.n) {
                pre[l] = a.posm[j];
                pre[l].w *= a.G;                                   // fold G into m_j
            } else {
                pre[l] = make_float4(kFarAway, kFarAway, kFarAway, 0.f);
            }
        }
    };
    auto store_tile = [&](int buf) {
#pragma unroll
        for (int l = 0; l < LPT; ++l) sj[buf][l * kThreads + tid] = pre[l];
    };

    if (t0 < t1) { load_tile(t0); store_tile(0); }
    __syncthreads();

    const f32x2 tiny2 = pk2(kTinyR2, kTinyR2);
    const f32x2 eps2 = pk2(a.eps, a.eps);

    for (int t = t0; t < t1; ++t) {
        const int buf = (t - t0) & 1;
        if (t + 1 < t1) load_tile(t + 1);            // global loads overlap the tile's math

        f32x2 ax[H], ay[H], az[H];
#pragma unroll
        for (int h = 0; h < H; ++h) ax[h] = ay[h] = az[h] = pk2(0.f, 0.f);

        float rc2 = 0.f;
        if (CONTACT) {
            const int jb = t * TJ, je = min(jb + TJ, a.n) - 1;
            const float Rj_max = (jb < a.n1 && je >= a.n1) ? fmaxf(R0, R1)
                                                           : star_radius(jb, a.n1, R0, R1);
            const float D = Ri_max + Rj_max;
            rc2 = D * D;
        }
        int qn = 0;                                  // candidate groups pushed in this tile

        const float4* __restrict__ s = sj[buf];
#pragma unroll 1
        for (int jg = 0; jg < TJ; jg += kGroupJ) {
            float rmin = 3.0e38f;
#pragma unroll
            for (int u_ = 0; u_ < kGroupJ; ++u_) {
                const float4 pj = s[jg + u_];            // LDS.128 broadcast
                const f32x2 xj = pk2(pj.x, pj.x), yj = pk2(pj.y, pj.y), zj = pk2(pj.z, pj.z);
#pragma unroll
                for (int h = 0; h < H; ++h) {
                    const f32x2 dx = add2(xj, nxi[h]);
                    const f32x2 dy = add2(yj, nyi[h]);
                    const f32x2 dz = add2(zj, nzi[h]);
                    f32x2 r2 = fma2(dx, dx, tiny2);
                    r2 = fma2(dy, dy, r2);
                    r2 = fma2(dz, dz, r2);
                    float r2l, r2h;
                    unpk2(r2, r2l, r2h);
                    const f32x2 y = pk2(rsqrt_approx(r2l), rsqrt_approx(r2h));   // 1/r
                    const f32x2 sft = fma2(r2, y, eps2);                           // r + eps
                    const f32x2 tt = mul2(sft, sft);                               // (r+eps)^2
                    float tl, th;
                    unpk2(tt, tl, th);
                    const float ipm = rcp_approx(tl * th) * pj.w;                  // one RCP for both lanes
                    const f32x2 um = pk2(ipm * th, ipm * tl);                      // G m_j/(r+eps)^2
                    const f32x2 c = mul2(um, y);                                   // G m_j/(r (r+eps)^2)  Eq. 4
                    ax[h] = fma2(c, dx, ax[h]);
                    ay[h] = fma2(c, dy, ay[h]);
                    az[h] = fma2(c, dz, az[h]);
                    if (CONTACT) rmin = fminf(rmin, fminf(r2l, r2h));              // FMNMX3
                }
            }
            if (CONTACT) {
                if (rmin < rc2) {                    // rare: one branch per kGroupJ elements j
                    queue[(qn & (kQueueDepth - 1)) * kThreads + tid] = (unsigned char)(jg / kGroupJ);
                    ++qn;
                }
            }
        }

#pragma unroll
        for (int h = 0; h < H; ++h) {
            float l, hgh;
            unpk2(ax[h], l, hgh); accx[2 * h] += (double)l; accx[2 * h + 1] += (double)hgh;
            unpk2(ay[h], l, hgh); accy[2 * h] += (double)l; accy[2 * h + 1] += (double)hgh;
            unpk2(az[h], l, hgh); accz[2 * h] += (double)l; accz[2 * h + 1] += (double)hgh;
        }

        if (CONTACT && qn > 0) {
            // Resolve this thread's candidate groups (the whole tile if the queue overflowed).
            const bool all = qn > kQueueDepth;
            const int cnt = all ? TJ / kGroupJ : qn;
#pragma unroll 1
            for (int q = 0; q < cnt; ++q) {
                const int jg = kGroupJ * (all ? q : (int)queue[q * kThreads + tid]);
#pragma unroll 1
                for (int jj = jg; jj < jg + kGroupJ; ++jj) {
                    const float4 pj = s[jj];
                    const int j = t * TJ + jj;
#pragma unroll
                    for (int h = 0; h < H; ++h) {
                        float xl, xh, yl, yh, zl, zh;
                        unpk2(nxi[h], xl, xh); unpk2(nyi[h], yl, yh); unpk2(nzi[h], zl, zh);
                        const float dxl = pj.x + xl, dyl = pj.y + yl, dzl = pj.z + zl;
                        const float dxh = pj.x + xh, dyh = pj.y + yh, dzh = pj.z + zh;
                        if (fmaf(dzl, dzl, fmaf(dyl, dyl, dxl * dxl)) < rc2)
                            contact_term(a, ibase + (2 * h) * kThreads, j, dxl, dyl, dzl, R0, R1,
                                         accx[2 * h], accy[2 * h], accz[2 * h]);
                        if (fmaf(dzh, dzh, fmaf(dyh, dyh, dxh * dxh)) < rc2)
                            contact_term(a, ibase + (2 * h + 1) * kThreads, j, dxh, dyh, dzh, R0, R1,
                                         accx[2 * h + 1], accy[2 * h + 1], accz[2 * h + 1]);
                    }
                }
            }
        }

        if (t + 1 < t1) store_tile(buf ^ 1);
        __syncthreads();
    }

    float4* __restrict__ out = a.part + (size_t)sp * a.n;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        const int i = ibase + k * kThreads;
        if (i < a.n) out[i] = make_float4((float)accx[k], (float)accy[k], (float)accz[k], 0.f);
    }
}

// ---------------------------------------------------------------------------
// Split-j reduction fused with the leapfrog update (rows a4 + a6 + a5).
//   a_i = sum_p src[p][i]  (fixed order, fp64)
//   if acc_out: acc_out[i] = a_i
//   v_i += kick_h * a_i ;  x_i += drift_dt * v_i        (either may be 0)
//   if advance: step += 1, R_s = ramp(step)             (expanding-star rule)
struct UpdateArgs {
    const float4* __restrict__ src;    // [nsrc][n]
    float4* acc_out;                   // may be null; may alias src when nsrc == 1
    float4* posm;
    float4* vel;
    DevState* dev;
    int n, nsrc;
    float kick_h, drift_dt;
    int advance;
};

__global__ void __launch_bounds__(256)
nb_reduce_update_kernel(const __grid_constant__ UpdateArgs u)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < u.n) {
        double sx = 0.0, sy = 0.0, sz = 0.0;
        for (int p = 0; p < u.nsrc; ++p) {
            const float4 q = u.src[(size_t)p * u.n + i];
            sx += (double)q.x; sy += (double)q.y; sz += (double)q.z;
        }
        const float ax = (float)sx, ay = (float)sy, az = (float)sz;
        if (u.acc_out) u.acc_out[i] = make_float4(ax, ay, az, 0.f);
        if (u.kick_h != 0.f || u.drift_dt != 0.f) {
            float4 v = u.vel[i];
            v.x = fmaf(u.kick_h, ax, v.x);
            v.y = fmaf(u.kick_h, ay, v.y);
            v.z = fmaf(u.kick_h, az, v.z);
            u.vel[i] = v;
            if (u.drift_dt != 0.f) {
                float4 p = u.posm[i];
                p.x = fmaf(u.drift_dt, v.x, p.x);
                p.y = fmaf(u.drift_dt, v.y, p.y);
                p.z = fmaf(u.drift_dt, v.z, p.z);
                u.posm[i] = p;
            }
        }
    }
    if (u.advance && blockIdx.x == 0 && threadIdx.x == 0) {
        DevState* d = u.dev;
        const long long nstep = d->step + 1;
        d->step = nstep;
        for (int s = 0; s < 2; ++s) {
            double Rs = d->R_start[s];
            if (d->n_ramp > 0) {
                const long long nn = nstep < d->n_ramp ? nstep : d->n_ramp;
                Rs = __dadd_rn(d->R_start[s],
                               __ddiv_rn(__dmul_rn(__dsub_rn(d->R_end[s], d->R_start[s]), (double)nn),
                                         (double)d->n_ramp));
            }
            d->R[s] = (float)Rs;
        }
    }
}

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

// Potential energies: per block, sum_i m_i * sum_{j != i} G m_j/(r+eps)  and
// sum_i sum_{j != i, contact} U_rep(r; R_ij)   (each unordered pair counted twice).
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
    for (int t = 0; t < njt; ++t) {
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
            const float w = (j == i) ? 0.f : pj.w;
            ph = fmaf(w, rcp_approx(r + a.eps), ph);
            if (a.gamma > 0.f && r2 < Dmax * Dmax && j != i && j < a.n) {
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

}  // namespace nb
