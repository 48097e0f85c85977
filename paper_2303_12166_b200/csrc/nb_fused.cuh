// nb_fused.cuh -- whole leapfrog steps of a SMALL system (n < 8,192) in one cooperative launch.
//
// At these sizes a step is a few microseconds of arithmetic (N = 2,048: 4.2e6 interactions) behind four or five
// dependent kernel launches, a stream fork and a join: the launches -- and the chain of memory latencies of a
// separate contact search -- are the step.  Here one persistent kernel runs rows a2-a6 of SURVEY.md 8(a) for any
// number of steps, its phases separated by grid-wide barriers:
//
//   [open]   v += dt/2 a ; x += dt v ; n += 1                     (nb_step: from the cached a(x_n))
//   repeat nforce times
//     F      the (i-block, j-split) work items of nb_gravity_kernel<2,128>: all-pairs gravity, Eq. 4
//            (PAPER.md:76), with the contact search INSIDE the loop: a pair whose fp32 r^2 is within reach of
//            R_i + R_j is queued and evaluated by contact_pair() in fp64 (Eqs. 5/6), its term
//            added to the same fp64 accumulators -- no contact slabs, no gather, no boxes.  (The big kernels
//            keep that test out of the N^2 loop because it costs ~10 % there; here nothing is ALU-bound.)
//     ---- grid barrier ----
//     U      a_i = sum of the j-split slabs (fixed order, fp64); kick, drift, n += 1; the last one is the
//            closing half kick and stores a(x) (nb_step), or stores a(x) only (nb_compute_accel)
//     ---- grid barrier ----
//
// One CTA per work item where they all fit (CTAs without work would spin in the barrier beside the working
// ones and slow them down), the elements of the update phase dealt round-robin to all CTAs.
// The step count and the radii live on the device (graph-safe): every thread reads n once at entry -- nobody
// writes it before the first barrier -- and follows it locally; thread 0 stores n and R_s(n) at the very end.
#pragma once
#include <cooperative_groups.h>
#include "nb_kernels.cuh"

namespace nb {

struct FusedArgs {
    GravArgs grav;             // slabs part[0 .. nsplit): gravity + contact terms of the j-split
    ContactArgs law;           // gamma (0: no contact terms), gamma_beta, v_dead, lens_mode
    float4* posm;              // state, updated in place
    float4* vel;
    float4* acc;               // cached acceleration a(x_n)
    float4* acc_out;           // nb_compute_accel: the caller's output as well (else nullptr)
    DevState* dev;
    int n, n1;
    float dt;
    int nforce;                // force evaluations (>= 1)
    int open;                  // 1: start with the opening half kick + drift from the cached acceleration
    int close_mode;            // 0: the last update is the closing half kick; 1: it stores a(x) and moves nothing
};

__global__ void __launch_bounds__(kThreads, 4)
nb_fused_step_kernel(const __grid_constant__ FusedArgs f)
{
    __shared__ float4 sj[2][128];
    __shared__ uint32_t queue_s[kInlineQueue][kThreads];
    __shared__ int pre_s[kThreads / 32][33];
    __shared__ double res_s[kThreads / 32][kInlineRound * 3];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const bool contact = f.law.gamma > 0.f;

    const long long step0 = f.dev->step, n_ramp = f.dev->n_ramp;
    const double Rs0 = f.dev->R_start[0], Rs1 = f.dev->R_start[1], Re0 = f.dev->R_end[0], Re1 = f.dev->R_end[1];
    long long nstep = step0;

    // one update phase: a_i from `nsrc` slabs of `src`, kick, drift.  Four lanes share an element: lane q adds up the
    // slabs q, q + 4, ... (one batch of loads in flight instead of four), then a fixed shuffle tree; the groups of
    // four are dealt round-robin to the CTAs so that all of them have work.
    auto update = [&](const float4* src, int nsrc, float4* out0, float4* out1, float kick_h, float drift_dt) {
        UpdateArgs u;
        u.acc64 = nullptr; u.src = src; u.acc_out = out0; u.posm = f.posm; u.vel = f.vel; u.dev = f.dev;
        u.n = f.n; u.nsrc = nsrc; u.kick_h = kick_h; u.drift_dt = drift_dt; u.vscale = 1.f; u.advance = 0;
        const int q = threadIdx.x & 3, g = threadIdx.x >> 2;                 // 32 groups of four lanes per CTA
        for (int i0 = 0; i0 < f.n; i0 += gridDim.x * (kThreads / 4)) {       // uniform trip count: the shuffles need all lanes
            const int i = i0 + blockIdx.x + gridDim.x * g;
            double sx = 0.0, sy = 0.0, sz = 0.0;
            if (i < f.n) {
#pragma unroll 4
                for (int s = q; s < nsrc; s += 4) {
                    const float4 t = src[(size_t)s * f.n + i];
                    sx += (double)t.x; sy += (double)t.y; sz += (double)t.z;
                }
            }
#pragma unroll
            for (int o = 2; o > 0; o >>= 1) {
                sx += __shfl_down_sync(0xffffffffu, sx, o);
                sy += __shfl_down_sync(0xffffffffu, sy, o);
                sz += __shfl_down_sync(0xffffffffu, sz, o);
            }
            if (i < f.n && q == 0) {
                float4 p, v;
                const float ax = (float)sx, ay = (float)sy, az = (float)sz;
                apply_update(u, i, ax, ay, az, p, v);
                if (out1) out1[i] = make_float4(ax, ay, az, 0.f);
            }
        }
    };

    if (f.open) {
        update(f.acc, 1, nullptr, nullptr, 0.5f * f.dt, f.dt);
        ++nstep;
        grid.sync();
    }

    const int G = f.grav.nib * f.grav.nsplit;
    for (int e = 0; e < f.nforce; ++e) {
        InlineContact ic;
        ic.law = &f.law; ic.vel = f.vel; ic.n1 = f.n1;
        ic.R0 = ramp_radius(Rs0, Re0, n_ramp, nstep); ic.R1 = ramp_radius(Rs1, Re1, n_ramp, nstep);
        ic.q = &queue_s[0][threadIdx.x]; ic.pre = &pre_s[0][0]; ic.res = &res_s[0][0];
        for (int item = blockIdx.x; item < G; item += gridDim.x) {
            if (contact) gravity_block<2, 128, true>(f.grav, item, sj, ic);
            else         gravity_block<2, 128, false>(f.grav, item, sj);
            __syncthreads();
        }
        grid.sync();
        if (e + 1 < f.nforce) {           // two half kicks merged: v += dt a ; x += dt v ; n += 1
            update(f.grav.part, f.grav.nsplit, nullptr, nullptr, f.dt, f.dt);
            ++nstep;
            grid.sync();
        } else if (f.close_mode == 0) {   // closing half kick; cache a(x_n)
            update(f.grav.part, f.grav.nsplit, f.acc, nullptr, 0.5f * f.dt, 0.f);
        } else {                          // a(x) only
            update(f.grav.part, f.grav.nsplit, f.acc, f.acc_out, 0.f, 0.f);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0 && nstep != step0) set_step(f.dev, nstep);
}

}  // namespace nb
