// nb_fused.cuh -- whole leapfrog steps of a SMALL system (n < 8,192) in one cooperative launch, ONE grid
// barrier per step.
//
// At these sizes a step is a few microseconds of arithmetic (N = 2,048: 4.2e6 interactions) behind four or five
// dependent kernel launches, a stream fork and a join: the launches -- and the chain of memory latencies of a
// separate contact search -- are the step.  Here one persistent kernel runs rows a2-a6 of SURVEY.md 8(a) for any
// number of steps.  Every CTA OWNS 2 P consecutive elements i (P packed pairs, a power of two chosen so that all
// CTAs are co-resident) and does everything for them:
//
//   [open]   own elements: v += dt/2 a ; x += dt v ; n += 1          (nb_step: from the cached a(x_n))
//            ---- grid barrier ----
//   repeat nforce times
//     S      ALL n positions (x, y, z, G m) staged in shared memory (16 B per element: <= 128 KB)
//     F      thread (pair p, segment s) walks the groups of 4 elements j  s, s + nseg, ...  for its two elements i:
//            all-pairs gravity, Eq. 4, with the contact search INSIDE the loop: a pair whose fp32 r^2
//            is within reach of R_i + R_j is queued and evaluated by contact_pair() in fp64 (Eqs. 5/6,
//            PAPER.md:80,84) -- the warp's queued pairs dealt evenly to its lanes -- and its term added to the
//            same fp64 accumulators.  (The big kernels keep that test out of the N^2 loop because it costs ~10 %
//            there; here nothing is ALU-bound.)
//     R      a_i = sum over the segments: a fixed shuffle butterfly inside the warp, then the CTA's 16 warps in
//            warp order through shared memory (fp64, bitwise reproducible) -- row a4 never leaves the CTA
//     U      own elements: kick, drift, n += 1; the last one is the closing half kick and stores a(x) (nb_step),
//            or stores a(x) only (nb_compute_accel)
//            ---- grid barrier ---- (not after the last)
//
// An earlier version split j over CTAs, which needed a second barrier per step (partial sums -> update phase)
// and ran a latency chain of 64 dependent group evaluations with one warp per scheduler: 13 us of a 19 us step
// was its force phase (config 1).
// Because a CTA updates its elements while others may still read them (the velocity of a contact partner), the
// state PING-PONGS between the caller's arrays and a scratch copy: a force evaluation reads one and writes the
// other.  The opening update (own elements only: safe either way) goes in place or across so that the LAST update
// lands in the caller's arrays.
// The step count and the radii live on the device (graph-safe): every thread reads n once at entry -- nobody
// writes it before the first barrier -- and follows it locally; thread 0 stores n and R_s(n) at the very end.
#pragma once
#include <cooperative_groups.h>
#include "nb_kernels.cuh"

namespace nb {

constexpr int kFusedGroup = 8;                     // elements j per group: four Montgomery pairs in flight per thread
constexpr int kFusedThreads = 512;                 // 16 warps: four per SM sub-partition
constexpr int kFusedWarps = kFusedThreads / 32;
constexpr int kFusedQueue = 16;                    // per-thread queue of (j, i slot) pairs that passed the fp32 pre-test
constexpr int kFusedRound = 32;                    // pairs a warp evaluates per round of the balanced evaluation
constexpr int kFusedMaxLogP = 5;                   // at most 32 packed pairs = 64 elements i per CTA
constexpr int kFusedFlush = 16;                    // groups of 8 j between flushes of the fp32 sums into fp64

struct FusedArgs {
    float4* posm;              // caller's state (buffer A), updated in place as seen from outside
    float4* vel;
    float4* posm2;             // scratch copy of the state (buffer B), [n] each
    float4* vel2;
    float4* acc;               // cached acceleration a(x_n)
    float4* acc_out;           // nb_compute_accel: the caller's output as well (else nullptr)
    DevState* dev;
    ContactArgs law;           // gamma (0: no contact terms), gamma_beta, v_dead, lens_mode
    int n, n1;
    float G, eps, dt;
    int nforce;                // force evaluations (>= 1)
    int open;                  // 1: start with the opening half kick + drift from the cached acceleration
    int close_mode;            // 0: the last update is the closing half kick; 1: it stores a(x) and moves nothing
    int relax;                 // 1: nb_relax (row f2, reading A17): the two half kicks of consecutive steps are NOT merged,
    float vscale;              //    the velocity is multiplied by vscale between them: v <- vscale (v + dt/2 a)
    int logP;                  // 2^logP packed pairs of elements i per CTA
    int npad;                  // n rounded up to a multiple of 8 (whole groups of elements j)
};

// Dynamic shared memory of the kernel for n elements.
inline size_t fused_smem_bytes(long long n)
{
    const size_t npad = (size_t)((n + kFusedGroup - 1) & ~(long long)(kFusedGroup - 1));
    return (npad + kFusedGroup) * sizeof(float4)                                   // positions + one far-away group
         + (size_t)kFusedQueue * kFusedThreads * sizeof(uint32_t)         // queues
         + (size_t)kFusedWarps * kFusedRound * 3 * sizeof(double)         // results of a round
         + (size_t)kFusedWarps * 64 * 3 * sizeof(double)                  // per-warp sums of the CTA's elements
         + (size_t)kFusedWarps * 34 * sizeof(int);                        // prefix counts
}

// Eq. 4 between the thread's packed pair of elements i and the 8 elements j at s[0..7] (x, y, z, G m): the
// arithmetic of gravity_group<1, false> (nb_kernels.cuh), but with NO branch inside -- the contact pre-test only
// sets a bit per (j, i slot) with fp32 r^2 <= thr, bit 2 u + slot -- so that ptxas interleaves the four
// independent rsqrt -> rcp chains (with a branch per pair of j a warp walked them one after the other, and a
// thread's 64 dependent evaluations were the force phase).
template <bool CON>
__device__ __forceinline__ unsigned fused_group(const float4* __restrict__ s, const f32x2 nx, const f32x2 ny, const f32x2 nz,
                                                const f32x2 eps2, f32x2& ax, f32x2& ay, f32x2& az, const float thr)
{
    const f32x2 tiny2 = pk2(kTinyR2, kTinyR2);
    unsigned mask = 0;
#pragma unroll
    for (int u = 0; u < kFusedGroup; u += 2) {
        const float4 p0 = s[u], p1 = s[u + 1];                     // LDS.128, broadcast within a segment
        const f32x2 dx0 = add2(pk2(p0.x, p0.x), nx), dy0 = add2(pk2(p0.y, p0.y), ny), dz0 = add2(pk2(p0.z, p0.z), nz);
        const f32x2 dx1 = add2(pk2(p1.x, p1.x), nx), dy1 = add2(pk2(p1.y, p1.y), ny), dz1 = add2(pk2(p1.z, p1.z), nz);
        f32x2 r20 = fma2(dx0, dx0, tiny2); r20 = fma2(dy0, dy0, r20); r20 = fma2(dz0, dz0, r20);
        f32x2 r21 = fma2(dx1, dx1, tiny2); r21 = fma2(dy1, dy1, r21); r21 = fma2(dz1, dz1, r21);
        float a0, b0, a1, b1;
        unpk2(r20, a0, b0); unpk2(r21, a1, b1);
        if (CON) {
            mask |= (a0 <= thr ? 1u : 0u) << (2 * u) | (b0 <= thr ? 1u : 0u) << (2 * u + 1)
                  | (a1 <= thr ? 1u : 0u) << (2 * u + 2) | (b1 <= thr ? 1u : 0u) << (2 * u + 3);
        }
        const f32x2 ri0 = pk2(rsqrt_approx(a0), rsqrt_approx(b0));     // 1/r
        const f32x2 ri1 = pk2(rsqrt_approx(a1), rsqrt_approx(b1));
        const f32x2 s0 = fma2(r20, ri0, eps2), s1 = fma2(r21, ri1, eps2);   // r + eps
        const f32x2 t0 = mul2(s0, s0), t1 = mul2(s1, s1);                   // (r + eps)^2
        const f32x2 Pt = mul2(t0, t1);
        float pl, ph;
        unpk2(Pt, pl, ph);
        const f32x2 iP = pk2(rcp_approx(pl), rcp_approx(ph));              // one RCP per two interactions
        const f32x2 k0 = mul2(mul2(t1, ri0), pk2(p0.w, p0.w)), k1 = mul2(mul2(t0, ri1), pk2(p1.w, p1.w));   // G m_j
        const f32x2 c0 = mul2(iP, k0), c1 = mul2(iP, k1);                  // G m_j / (r (r+eps)^2)  Eq. 4
        ax = fma2(c0, dx0, ax); ay = fma2(c0, dy0, ay); az = fma2(c0, dz0, az);
        ax = fma2(c1, dx1, ax); ay = fma2(c1, dy1, ay); az = fma2(c1, dz1, az);
    }
    return mask;
}

__global__ void __launch_bounds__(kFusedThreads, 1)
nb_fused_step_kernel(const __grid_constant__ FusedArgs f)
{
    extern __shared__ float4 fused_smem[];
    float4* __restrict__ sx = fused_smem;                                                  // [npad + 8]
    uint32_t* __restrict__ queue = reinterpret_cast<uint32_t*>(sx + f.npad + kFusedGroup);           // [kFusedQueue][512]
    double* __restrict__ res = reinterpret_cast<double*>(queue + kFusedQueue * kFusedThreads);   // [16][kFusedRound * 3]
    double* __restrict__ red = res + kFusedWarps * kFusedRound * 3;                        // [16][64][3]
    int* __restrict__ pre = reinterpret_cast<int*>(red + kFusedWarps * 64 * 3);            // [16][34]

    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int P = 1 << f.logP, ip = tid & (P - 1), seg = tid >> f.logP, nseg = kFusedThreads >> f.logP;
    const int base = blockIdx.x * 2 * P;               // the CTA's elements: base ... base + 2 P - 1
    const int e0 = base + 2 * ip;                      // the thread's two elements i: e0, e0 + 1
    const int eu = base + tid;                         // the element this thread updates (tid < 2 P)
    const bool contact = f.law.gamma > 0.f;
    const int n = f.n;

    const long long step0 = f.dev->step, n_ramp = f.dev->n_ramp;
    const double Rs0 = f.dev->R_start[0], Rs1 = f.dev->R_start[1], Re0 = f.dev->R_end[0], Re1 = f.dev->R_end[1];
    long long nstep = step0;

    // where the state is (read) and where the next update puts it
    float4 *xs = f.posm, *vs = f.vel, *xd = f.posm2, *vd = f.vel2;
    auto swap_buffers = [&]() { float4* t = xs; xs = xd; xd = t; t = vs; vs = vd; vd = t; };

    // element eu, given a: v += kick_h a ; [v *= scale ; v += kick2_h a] ; x += drift_dt v, read from (xs, vs),
    // written to (xo, vo)
    auto move = [&](float ax, float ay, float az, float kick_h, float drift_dt, float4* xo, float4* vo,
                    bool damp = false, float kick2_h = 0.f) {
        float4 v = __ldcg(vs + eu), p = __ldcg(xs + eu);
        v.x = fmaf(kick_h, ax, v.x); v.y = fmaf(kick_h, ay, v.y); v.z = fmaf(kick_h, az, v.z);
        if (damp) {
            if (f.vscale != 1.f) { v.x *= f.vscale; v.y *= f.vscale; v.z *= f.vscale; }
            if (kick2_h != 0.f) { v.x = fmaf(kick2_h, ax, v.x); v.y = fmaf(kick2_h, ay, v.y); v.z = fmaf(kick2_h, az, v.z); }
        }
        if (drift_dt != 0.f) {
            p.x = fmaf(drift_dt, v.x, p.x); p.y = fmaf(drift_dt, v.y, p.y); p.z = fmaf(drift_dt, v.z, p.z);
        }
        vo[eu] = v; xo[eu] = p;
    };

    const int moves = f.close_mode == 0 ? f.nforce : f.nforce - 1;     // updates that ping-pong the state
    if (f.open) {
        const bool across = (moves & 1) != 0;          // so that the last update lands in the caller's arrays
        if (tid < 2 * P && eu < n) {
            const float4 a = f.acc[eu];
            move(a.x, a.y, a.z, 0.5f * f.dt, f.dt, across ? xd : xs, across ? vd : vs);
        }
        if (across) swap_buffers();
        ++nstep;
        grid.sync();
    }

    const int ngroups = f.npad / kFusedGroup;
    const int K = (ngroups + nseg - 1) / nseg;         // groups per thread (the same for all: the warp stays together)
    const f32x2 eps2 = pk2(f.eps, f.eps);
    uint32_t* __restrict__ q = queue + tid;            // the thread's queue: q[k * kFusedThreads]

    for (int e = 0; e < f.nforce; ++e) {
        const bool last = e + 1 == f.nforce;
        const float R0 = ramp_radius(Rs0, Re0, n_ramp, nstep), R1 = ramp_radius(Rs1, Re1, n_ramp, nstep);

        // S: all positions -> shared memory, G folded into the mass
#pragma unroll 4
        for (int j = tid; j < f.npad + kFusedGroup; j += kFusedThreads) {        // (unrolled: four loads in flight per thread)
            float4 p = make_float4(kFarAway, kFarAway, kFarAway, 0.f);
            if (j < n) { p = __ldcg(xs + j); p.w *= f.G; }
            sx[j] = p;
        }
        // what contact_pair() needs of the thread's own elements beyond the staged positions: (v, m) and R
        const int i0 = min(e0, f.npad), i1 = min(e0 + 1, f.npad);       // index npad is a far-away dummy
        float4 cvi[2];
        float Ri[2] = {0.f, 0.f};
#pragma unroll
        for (int l = 0; l < 2; ++l) {
            cvi[l] = make_float4(0.f, 0.f, 0.f, 1.f);
            if (contact && e0 + l < n) {
                const float4 w = __ldcg(vs + e0 + l);
                cvi[l] = make_float4(w.x, w.y, w.z, __ldcg(&xs[e0 + l].w));
                Ri[l] = star_radius(e0 + l, f.n1, R0, R1);
            }
        }
        __syncthreads();

        // F: gravity over the thread's groups of elements j, contact candidates queued
        const float4 pa = sx[i0], pb = sx[i1];
        f32x2 nxi[1] = {pk2(-pa.x, -pb.x)}, nyi[1] = {pk2(-pa.y, -pb.y)}, nzi[1] = {pk2(-pa.z, -pb.z)};
        const float Rm = fmaxf(Ri[0], Ri[1]), Rmax = fmaxf(R0, R1);
        double accx[2] = {0.0, 0.0}, accy[2] = {0.0, 0.0}, accz[2] = {0.0, 0.0};
        f32x2 ax[1] = {pk2(0.f, 0.f)}, ay[1] = {pk2(0.f, 0.f)}, az[1] = {pk2(0.f, 0.f)};
        int nq = 0;

        auto flush = [&]() {                         // fp32 sums of <= 128 terms -> fp64
            float l, h;
            unpk2(ax[0], l, h); accx[0] += (double)l; accx[1] += (double)h;
            unpk2(ay[0], l, h); accy[0] += (double)l; accy[1] += (double)h;
            unpk2(az[0], l, h); accz[0] += (double)l; accz[1] += (double)h;
            ax[0] = ay[0] = az[0] = pk2(0.f, 0.f);
        };
        // one queued pair (i, j) as the acceleration it gives i, fp64
        auto pair_accel = [&](int i, int j, const float4 vi, float Rii, double& fx, double& fy, double& fz) {
            const float4 xi = sx[i], xj = sx[j], vj = __ldcg(vs + j);
            contact_pair(f.law, make_float4(xi.x, xi.y, xi.z, Rii), vi,
                         make_float4(xj.x, xj.y, xj.z, star_radius(j, f.n1, R0, R1)), vj, fx, fy, fz);
            const double im = 1.0 / (double)vi.w;
            fx *= im; fy *= im; fz *= im;
        };
        auto drain = [&]() {                         // the thread's own queue, in the order found (nearly full: dense overlaps)
            for (int h = 0; h < nq; ++h) {
                const uint32_t w = q[h * kFusedThreads];
                const int j = (int)(w >> 4), l = (int)(w & 1u), i = e0 + l;
                if (j >= n || i >= n || j == i) continue;
                double fx, fy, fz;
                pair_accel(i, j, l ? cvi[1] : cvi[0], l ? Ri[1] : Ri[0], fx, fy, fz);
                if (l) { accx[1] += fx; accy[1] += fy; accz[1] += fz; }
                else   { accx[0] += fx; accy[0] += fy; accz[0] += fz; }
            }
            nq = 0;
        };

#pragma unroll 1
        for (int k = 0; k < K; ++k) {
            int g = seg + k * nseg;
            if (g >= ngroups) g = ngroups;           // the far-away group: contributes exactly 0
            const int j0 = g * kFusedGroup;
            if (contact) {
                const float Rj = j0 + kFusedGroup - 1 < f.n1 ? R0 : (j0 >= f.n1 ? R1 : Rmax);
                const float D = Rm + Rj;
                const float thr = D * D * (1.0f + 1.0e-5f) + kTinyR2;
                unsigned mask = fused_group<true>(sx + j0, nxi[0], nyi[0], nzi[0], eps2, ax[0], ay[0], az[0], thr);
                while (mask) {                       // within reach of a contact (or the self pair): queue for the fp64 test
                    const int b = __ffs((int)mask) - 1;
                    mask &= mask - 1;
                    if (nq == kFusedQueue) drain();
                    q[(nq++) * kFusedThreads] = ((uint32_t)(j0 + (b >> 1)) << 4) | (uint32_t)(b & 1);
                }
            } else {
                fused_group<false>(sx + j0, nxi[0], nyi[0], nzi[0], eps2, ax[0], ay[0], az[0], -1.f);
            }
            if ((k & (kFusedFlush - 1)) == kFusedFlush - 1) flush();
        }
        flush();

        if (contact) {
            // the warp's queued pairs dealt evenly to its lanes -- a lane with 6 pairs no longer holds up 31 lanes
            // with 1 -- evaluated, and handed back through shared memory; every lane adds ITS pairs in the order found
            int inc = nq;
            for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
            const int total = __shfl_sync(0xffffffffu, inc, 31), mine0 = inc - nq;
            int* __restrict__ pw = pre + warp * 34;
            double* __restrict__ rw = res + warp * (kFusedRound * 3);
            pw[lane] = mine0;
            if (lane == 31) pw[32] = total;
            __syncwarp();
            for (int p0 = 0; p0 < total; p0 += kFusedRound) {
                const int pe = min(total, p0 + kFusedRound);
                for (int p = p0 + lane; p < pe; p += 32) {
                    int lo = 0;                      // owner: the largest lane with pre[lane] <= p
#pragma unroll
                    for (int s2 = 16; s2 > 0; s2 >>= 1) if (pw[lo + s2] <= p) lo += s2;
                    const int ot = tid - lane + lo;
                    const uint32_t w = queue[(p - pw[lo]) * kFusedThreads + ot];
                    const int j = (int)(w >> 4), i = base + 2 * (ot & (P - 1)) + (int)(w & 1u);
                    double fx = 0.0, fy = 0.0, fz = 0.0;
                    if (j < n && i < n && j != i) {
                        const float4 wi = __ldcg(vs + i);
                        pair_accel(i, j, make_float4(wi.x, wi.y, wi.z, __ldcg(&xs[i].w)), star_radius(i, f.n1, R0, R1), fx, fy, fz);
                    }
                    rw[(p - p0) * 3] = fx; rw[(p - p0) * 3 + 1] = fy; rw[(p - p0) * 3 + 2] = fz;
                }
                __syncwarp();
                const int b = max(mine0, p0), en = min(mine0 + nq, pe);
                for (int p = b; p < en; ++p) {
                    const double fx = rw[(p - p0) * 3], fy = rw[(p - p0) * 3 + 1], fz = rw[(p - p0) * 3 + 2];
                    if (q[(p - mine0) * kFusedThreads] & 1u) { accx[1] += fx; accy[1] += fy; accz[1] += fz; }
                    else                                     { accx[0] += fx; accy[0] += fy; accz[0] += fz; }
                }
                __syncwarp();
            }
        }

        // R: sum over the segments.  Lanes with the same pair index: xor butterfly (the same tree in every lane,
        // operands commuted: the same bits); then the CTA's 16 warps in warp order.
        for (int o = 16; o >= P; o >>= 1) {
#pragma unroll
            for (int l = 0; l < 2; ++l) {
                accx[l] += __shfl_xor_sync(0xffffffffu, accx[l], o);
                accy[l] += __shfl_xor_sync(0xffffffffu, accy[l], o);
                accz[l] += __shfl_xor_sync(0xffffffffu, accz[l], o);
            }
        }
        if (lane < P) {                              // lane == pair index here
#pragma unroll
            for (int l = 0; l < 2; ++l) {
                double* __restrict__ r = red + ((size_t)warp * 64 + 2 * lane + l) * 3;
                r[0] = accx[l]; r[1] = accy[l]; r[2] = accz[l];
            }
        }
        __syncthreads();
        if (tid < 2 * P && eu < n) {
            double sxx = 0.0, syy = 0.0, szz = 0.0;
#pragma unroll
            for (int w = 0; w < kFusedWarps; ++w) {
                const double* __restrict__ r = red + ((size_t)w * 64 + tid) * 3;
                sxx += r[0]; syy += r[1]; szz += r[2];
            }
            const float fax = (float)sxx, fay = (float)syy, faz = (float)szz;
            // U
            if (!last) {
                if (f.relax) move(fax, fay, faz, 0.5f * f.dt, f.dt, xd, vd, true, 0.5f * f.dt);   // half kick, damp, half kick, drift
                else         move(fax, fay, faz, f.dt, f.dt, xd, vd);   // two half kicks merged: v += dt a ; x += dt v
            } else if (f.close_mode == 0) {          // closing half kick (nb_relax: then v <- vscale v); cache a(x_n)
                move(fax, fay, faz, 0.5f * f.dt, 0.f, xd, vd, f.relax != 0);
                f.acc[eu] = make_float4(fax, fay, faz, 0.f);
            } else {                                 // a(x) only
                f.acc[eu] = make_float4(fax, fay, faz, 0.f);
                if (f.acc_out) f.acc_out[eu] = make_float4(fax, fay, faz, 0.f);
            }
        }
        if (!last) {
            swap_buffers();
            ++nstep;
            grid.sync();
        }
    }
    if (blockIdx.x == 0 && tid == 0 && nstep != step0) set_step(f.dev, nstep);
}

}  // namespace nb
