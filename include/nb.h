/*
 * nb.h -- C ABI of the B200-native all-pairs binary-star element model.
 *
 * The hot path of arXiv 2303.12166 ("N-body simulation of binary star mass
 * transfer using NVIDIA GPUs"): the O(N^2) pair-wise element-to-element
 * acceleration (Eqs. 4-6; "the sum total of all the pair-wise
 * element to element interactions") and the leapfrog step that
 * consumes it, with the per-star expanding element radius
 * (PAPER.md:60,89).  Every step of the path runs in hand-written sm_100a CUDA
 * kernels (paper_2303_12166_b200/csrc); there is no CPU fallback.
 *
 * Conventions
 *   - Every function returns NB_OK (0) or a negative nb_status; nothing aborts
 *     or throws.  nb_strerror() gives the text; for NB_ECUDA, nb_last_cuda_error()
 *     gives the cudaError_t.
 *   - "dev" pointers are CUDA device pointers on the device that was current
 *     at nb_create(); "host" pointers are ordinary host memory.  That device must
 *     be current in every later call on the ctx (NB_ESTATE otherwise).
 *   - The CALLER owns every device byte (state, output, workspace).  The
 *     library owns only the host-side nb_ctx (plus one internal stream and two events: SURVEY 8(b) says
 *     "owns only the host-side nb_ctx" -- the stream carries the contact pass beside the gravity kernel and
 *     is created and destroyed with the ctx) and never allocates device memory.
 *     Borrowed pointers must stay valid until the next nb_set_state()/nb_destroy().
 *   - All device work is ordered on the borrowed stream given to nb_create() (the contact
 *     pass runs on a library-owned non-blocking stream, forked from and joined back into the
 *     borrowed stream by events inside each force evaluation -- invisible to the caller).
 *     Nothing synchronises except nb_set_state() (SURVEY 8(b) lists only nb_energy(); binding has to
 *     read back the verdict on star[] before it can return NB_ESTATE), nb_energy(), nb_get_step(),
 *     nb_transfer_diagnostics() and nb_download_state().  One ctx per host thread.
 *   - Element layout: elements of star 0 first, then star 1.  posm[i] =
 *     (x, y, z, m_i), vel[i] = (vx, vy, vz, unused); both float4, 16-byte aligned.
 *
 * Model (readings A1-A16 are listed in DESIGN.md):
 *   d = x_j - x_i, r = |d|, R_ij = (R_star(i) + R_star(j))/2
 *   a_i = sum_{j != i, r > 0} [ G m_j/(r+eps)^2 - (in contact: g*pi*V(r;R_ij)/m_i) ] d/r
 *   in contact  <=> gamma > 0 and r < 2 R_ij
 *   V(r;R) = 4/3 R^3 - R^2 r + r^3/12   (lens_mode 0: displaced volume, A1)
 *          = 4/3 R^3 - R^2 r + r^2/12   (lens_mode 1: as printed)
 *   g = gamma        if d.(v_j - v_i)/r < -v_dead   (converging, Eq. 5)
 *     = gamma*beta   otherwise                      (diverging,  Eq. 6)
 *   R_s(n) = R_start[s] + (R_end[s]-R_start[s]) * min(n, n_ramp)/n_ramp
 *   step:  kick-drift-kick leapfrog, one force evaluation per step, a(x_{n+1})
 *          evaluated with the half-step velocity (A7).
 */
#ifndef NB_H_
#define NB_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nb_ctx nb_ctx;

typedef enum {
    NB_OK = 0,
    NB_EINVAL = -1,   /* bad argument (null, n out of range, misaligned, bad parameter) */
    NB_ESTATE = -2,   /* call order (no state set), or star[] not 0...0 1...1 */
    NB_ECUDA = -3,    /* a CUDA call failed; see nb_last_cuda_error() */
    NB_ENOMEM = -4,   /* workspace too small / host allocation failed */
    NB_EARCH = -5,    /* the current device is not sm_100 */
    NB_ESIZE = -6     /* n exceeds the fixed scratch of nb_gravity_accel_static() (see its limit) */
} nb_status;

typedef struct {
    float G, eps, dt, q;        /* Eq. 4 G and eps; leapfrog step (89);
                                   q = m2/m1 in (0,1] -- validated, metadata */
    float gamma, beta;          /* Eqs. 5/6; gamma = 0 disables contact
                                   terms; 0 < beta <= 1 */
    float R_start[2], R_end[2]; /* element radius per star: expanding-star rule
                                   (PAPER.md:89); equal => static */
    int32_t n_ramp;             /* steps over which R goes start->end; 0 => R = R_start */
    float v_dead;               /* converging iff rdot < -v_dead; 0 = literal rule (A5) */
    int32_t lens_mode;          /* 0: r^3/12 displaced volume (A1); 1: r^2/12 as printed */
} nb_params;

/* Create a context for up to n_max elements.  `cuda_stream` is a cudaStream_t
 * (NULL = the legacy default stream), borrowed.  Fails with NB_EARCH unless the
 * current device has compute capability 10.x. */
int nb_create(nb_ctx** out, int64_t n_max, const nb_params* p, void* cuda_stream);

/* Bytes of device workspace nb_set_state() needs for a context of n_max elements: cached acceleration,
 * the gravity kernel's partial sums (slabs of n float4 for n < 98304; from there on the symmetric kernel adds
 * into two fp64 sums per element instead), device-side step/radius state, reduction scratch, and the contact
 * pass's cell table, counting-sort buffers and ordered copy.  3 MiB at n_max = 2048, 134 MiB at 65536,
 * 322 MiB at 262144, 419 MiB at 1048576.  0 if n_max is out of range. */
size_t nb_workspace_bytes(int64_t n_max);

/* Bind the state.  posm, vel: dev float[n][4], 16-byte aligned, BORROWED and
 * updated in place by nb_step().  star: dev int32[n], values 0...0 1...1 (checked
 * on the device; read only during this call).  workspace: dev, 256-byte aligned,
 * >= nb_workspace_bytes(n_max) bytes, BORROWED.  Resets the step count to 0 and
 * drops the cached acceleration.  Synchronises the stream.  1 <= n <= n_max. */
int nb_set_state(nb_ctx* ctx, int64_t n, float* posm, float* vel, const int32_t* star,
                 void* workspace, size_t workspace_bytes);

/* One evaluation of Eqs. 4-6 at the current (x, v, R(n)).  acc: dev float[n][4],
 * caller-owned output, receives (ax, ay, az, 0).  Asynchronous on the stream. */
int nb_compute_accel(nb_ctx* ctx, float* acc);

/* nsteps leapfrog steps, asynchronous on the stream.  On
 * completion of the stream work posm/vel hold (x_{n+nsteps}, v_{n+nsteps}),
 * velocities synchronised with positions.  nsteps >= 0. */
int nb_step(nb_ctx* ctx, int nsteps);

/* Diagnostics at the current state, written to HOST out[12]:
 * KE, U_grav, U_rep, E, Px, Py, Pz, Lx, Ly, Lz, |sum m_i a_i|, step count.
 * U_grav = -sum_{i<j} G m_i m_j/(r+eps); U_rep per A12.  Synchronises the stream. */
int nb_energy(nb_ctx* ctx, double* out);

/* ---- SURVEY.md 8(f) "next" rows: built on the same state, kernels and stream ---------------
 *
 * f2, star construction (elements are put together and "this technique was used to
 * create a binary system"; no procedure is printed -- reading A17): nsteps leapfrog steps as in
 * nb_step(), each followed by v <- max(0, 1 - kappa*dt) v, so a star (or the binary) settles
 * into equilibrium.  kappa >= 0 [1/time]; kappa = 0 is nb_step() up to fp32 rounding (nb_step merges the two
 * half kicks of consecutive steps into one multiply-add, nb_relax cannot).  The step count and the
 * radius ramp advance as usual.  Asynchronous on the stream. */
int nb_relax(nb_ctx* ctx, int nsteps, float kappa);

/* f3, mass transfer through L1 (reading A18), written to HOST out[32]:
 *   [0] M0 [1] M1   masses of the two stars by membership;  [18..23] centres X0, X1;  [24..29] V0, V1
 *   [2] a = |X1 - X0|   [3] d0: distance of the L1 plane from X0 along e = (X1 - X0)/a
 *   [4] rL0 [5] rL1   Roche-lobe radii, a * Eq. 3 (constant k_lobe: 0.6 standard, 0.69 as printed, A9)
 *   [6] Mcross0 [7] Mcross1   mass of star s's elements beyond the L1 plane (on the other star's side)
 *   [8] Min0 [9] Min1         ... inside the OTHER star's lobe sphere |x - X_o| < rL_o
 *   [10] Mout0 [11] Mout1     ... outside both lobe spheres
 *   [12..14] Ldisk0 [15..17] Ldisk1   angular momentum of the Min_s elements about the other star,
 *                                     sum m (x - X_o) x (v - V_o)
 *   [30] step count, [31] 0.
 * All sums and decisions in fp64 on the fp32 state, all of them on the device (star centres, the L1 plane by
 * Newton iteration on the force balance, Eq. 3); the record is then copied to the host.  Synchronises the stream. */
int nb_transfer_diagnostics(nb_ctx* ctx, double k_lobe, double* out);

/* f3 per step, on the device ("donor mass beyond the L1 plane / inside the accretor's lobe per step";
 * PAPER.md:15, 107-109): the same 32-double record, written to row n of dev_series[rows][32] (DEVICE memory,
 * caller-owned, 8-byte aligned), n = the run's step count when the launches execute; a run past the last row
 * (n >= rows) writes nothing.  Four short launches on the ctx stream, no host synchronisation: call it after
 * nb_step(1) in a loop (or capture the pair in a CUDA graph) and read the series back once at the end.
 * Rows the run did not visit keep whatever the caller put there. */
int nb_transfer_record(nb_ctx* ctx, double k_lobe, double* dev_series, int64_t rows);

/* f4, headless point splat in place of the paper's OpenGL viewer (reading A19):
 * orthographic projection of the element positions on coordinate axes (axis_u, axis_v in {0,1,2},
 * different), window centred at HOST centre[3] with half width half_width along u (square pixels
 * of 2*half_width/W), pixel = floor((x - c) * W/(2*half_width) + W/2 resp. H/2) evaluated in
 * float32 with one rounding per operation.  image: dev uint32[2][H][W], caller-owned, overwritten
 * with the number of elements of each star per pixel (exact, integer atomics).  Asynchronous. */
int nb_splat(nb_ctx* ctx, const float* centre, float half_width, int axis_u, int axis_v, int W, int H,
             uint32_t* image);

/* Current step count n and element radii R_s(n) (host outputs; either may be NULL).
 * Synchronises the stream. */
int nb_get_step(nb_ctx* ctx, int64_t* step, float* R);

/* Restore the step count n of a checkpointed run (the element radius is a function of
 * how far the run has come): sets n = step and R_s(n) by the expanding-star rule, exactly as nsteps
 * calls of nb_step() from 0 would have left them.  The full state of a run is (x, v, a(x_n), n):
 * nb_upload_state() restores the arrays, this call the count.  A cached acceleration that came with
 * nb_upload_state(host_acc) is kept (it belongs to the uploaded state: upload first, then set the step).
 * One evaluated by this ctx (nb_compute_accel, nb_step, ...) holds contact terms at the OLD radii: it is
 * dropped when the radii move with the step count (gamma > 0, n_ramp > 0, R_start != R_end), and the next
 * step evaluates a(x) again at R_s(step).  step >= 0.  Asynchronous on the stream. */
int nb_set_step(nb_ctx* ctx, int64_t step);

/* Host-buffer entry points for end-to-end use and checkpoint/restart: copy HOST
 * float[n][4] arrays into / out of the bound device buffers on the ctx stream.
 * The full state of a run is (x, v, a(x_n), n): host_acc carries the cached
 * acceleration (the one the next nb_step() starts from, which saw the half-step
 * velocity, A7).  Upload with host_acc == NULL drops the cache, so the next step
 * re-evaluates a(x_n) with the uploaded velocities; the step count is kept.
 * Download with host_acc != NULL evaluates a(x_n) first if it is not cached.
 * Download synchronises the stream.  Pinned host memory makes the copies
 * asynchronous.  Any pointer may be NULL (skipped). */
int nb_upload_state(nb_ctx* ctx, const float* host_posm, const float* host_vel, const float* host_acc);
int nb_download_state(nb_ctx* ctx, float* host_posm, float* host_vel, float* host_acc);

/* Launch configuration chosen for the bound state (for reports): i-elements per
 * CTA, j-splits P, CTAs of the force kernel, CTAs of the update kernel (one-sided kernel);
 * super-tile size S, super-tiles T (= partial-sum slabs), CTAs = T(T+1)/2, CTAs of the update
 * kernel (symmetric kernel); elements i per CTA, j segments per CTA, CTAs, CTAs (n < 8192: the
 * one cooperative launch that runs whole steps). */
int nb_get_launch_info(nb_ctx* ctx, int32_t* out4);

/* Which kernel evaluates row a2 (Eq. 4, summed over all pairs).
 *   NB_PATH_AUTO (default): the symmetric kernel for n >= 8192; for n < 8192 the one-sided loop inside
 *     nb_fused_step_kernel: ONE cooperative launch per nb_step() / nb_relax() / nb_compute_accel() call runs
 *     rows a2-a6 for all its steps (every CTA owns a slice of elements i; the state ping-pongs between the
 *     caller's arrays and workspace scratch inside the launch and is back in the caller's arrays at its end).
 *     NB_PATH_ONE_SIDED takes the same launch for n < 8192.
 *   NB_PATH_ONE_SIDED: every ORDERED pair (i, j) is evaluated; a CTA owns an (i-block, j-split).
 *   NB_PATH_SYMMETRIC: every UNORDERED pair is evaluated once and serves both a_i and a_j
 *     (the force of Eq. 4 is "between elements i and j": F_ij = -F_ji); a CTA owns a pair of
 *     super-tiles.  Both compute the same sum in a fixed order (bitwise reproducible run to run);
 *     they differ from each other by fp32 rounding only.
 * May be called before or after nb_set_state(); NB_ENOMEM if the bound workspace cannot hold the
 * partial sums of the requested path for the bound n (it always can for the default path).  Drops nothing: the
 * cached acceleration stays valid.
 * For n >= 98304 the symmetric kernel runs in "chain mode": its CTAs add their results into one pair of fp64 sums per
 * element, super-tile by super-tile in a fixed order kept by turn counters (still bitwise reproducible, no atomics
 * on data).  Should a turn ever fail to come (it cannot by construction; the check keeps a bug from hanging the GPU),
 * an error word is raised on the device that only nb_set_state() clears: every synchronising call from then on
 * (nb_energy, nb_get_step, nb_download_state) returns NB_ECUDA with nb_last_cuda_error() == cudaErrorLaunchTimeout
 * and drops the cached acceleration -- the state has been stepped with sums added out of order; rebind it. */
enum { NB_PATH_AUTO = 0, NB_PATH_ONE_SIDED = 1, NB_PATH_SYMMETRIC = 2 };
int nb_set_force_path(nb_ctx* ctx, int path);

/* Name (template instantiation) of the row-a2 kernel chosen for the bound state, for reports;
 * "" if no state is bound.  The string is static. */
const char* nb_force_kernel_name(nb_ctx* ctx);

/* Kernels launched by this ctx since nb_create() (for bench accounting). */
int64_t nb_launch_count(nb_ctx* ctx);

/* Measurement aids: launch the all-pairs gravity kernel (row a2: Eq. 4 over all N^2 ordered
 * pairs; nb_time_force_kernel) or the contact pass (row a3: cell list -- bbox, count, scan, scatter, rank -- and Eqs. 5/6;
 * nb_time_contact_pass, 0 ms when gamma == 0) `reps` times on the ctx stream after one warm-up,
 * bracketed by CUDA events on that stream; HOST *ms_avg receives the average duration of one
 * pass.  Their partial sums land in the workspace and touch no state (in chain mode, n >= 98304, the
 * gravity launches overwrite the fp64 accumulators of the last force evaluation -- the cached acceleration
 * is a separate array and stays valid -- and leave the chain error word alone).  Synchronise the stream. */
int nb_time_force_kernel(nb_ctx* ctx, int reps, float* ms_avg);
int nb_time_contact_pass(nb_ctx* ctx, int reps, float* ms_avg);

/* Measurement aid for row a3: one contact pass (which pairs are "in contact") in counting mode.
 * HOST out2[0] = candidate pairs the search pre-tests (ordered: each element against the elements of the cells of
 * its query), out2[1] = pairs that pass the fp32 pre-test and are evaluated in fp64 (about twice the number of
 * unordered contacts).  n < 8192 (no cell list): out2[0] = n (n - 1), out2[1] = -1.  gamma == 0: zeros.
 * The partial sums it writes touch no state.  Synchronises the stream. */
int nb_contact_stats(nb_ctx* ctx, int64_t* out2);

/* ---- Gravity accelerations for callers that cannot allocate device memory ------------------------------
 *
 * Everything above needs a workspace the caller has to get from somewhere (3 MiB at n = 2048), plus a ctx
 * whose creation makes a stream and two events.  Some users of this library have no way to obtain that
 * memory: code loaded as a plug-in into a host application that hands it exactly the state arrays and keeps
 * its allocator to itself, code running under a fixed, fully assigned memory budget, and code inside a
 * latency-critical loop where cudaMalloc/cudaFree are off limits because they stall the whole device.
 * For them this one call evaluates row a2 -- Eq. 4 summed over all pairs,
 *   a_i = sum_{j != i} G m_j d / (r (r + eps)^2),  d = x_j - x_i,  r = |d|  (coincident pairs add nothing) --
 * with the one-sided all-pairs kernel (NB_PATH_ONE_SIDED above) and needs nothing but its inputs and its
 * output: the kernel's scratch (the partial sums of its j splits, which a second kernel adds up in split
 * order) lives in a fixed array inside the library image instead of a workspace.  No ctx, no contact terms
 * (gamma = 0), no stepping.
 *
 *   posm: dev float[n][4] (x, y, z, m), 16-byte aligned, read only.   acc: dev float[n][4], 16-byte aligned,
 *   receives (ax, ay, az, 0); must not overlap posm.   cuda_stream: cudaStream_t (NULL = legacy default
 *   stream); the two launches are asynchronous on it.   cuda_error: HOST, may be NULL; receives the
 *   cudaError_t when the call returns NB_ECUDA, else 0.
 *
 * Limit: 1 <= n <= nb_gravity_accel_static_max_n() = 16384.  A larger n returns NB_ESIZE and launches
 * nothing -- use the ctx API with a caller-provided workspace there.
 *
 * Costs and rules that follow from the fixed array:
 *   - it is 2 MiB (131072 float4) of device memory on EVERY GPU this process uses the library on, held
 *     from the moment the library is loaded there until the process exits, whether or not this is called;
 *   - the call itself performs no cudaMalloc, no cudaFree, creates no stream or event and calls no library
 *     routine that allocates;
 *   - the first call on a device looks up the array's device address (once per device, with that device
 *     current) and the device's SM count and compute capability; later calls on that device reuse them.
 *     Make that first call before you begin any stream capture;
 *   - every call on a device uses the same array, and it still holds the previous call's partial sums
 *     when the next one starts.  Nothing has to be zeroed: each call writes every slot before it reads it.
 *     But two calls whose kernels are in flight on the same device at once (different streams, or
 *     different host threads) overwrite each other's partial sums -- the results of both are garbage and
 *     nothing reports it.  Keep all calls on one device on one stream, or order them with events.
 * Returns NB_EINVAL (null/misaligned pointer, n < 1, G or eps negative or not finite), NB_ESIZE, NB_EARCH
 * (device is not sm_100), NB_ECUDA, else NB_OK.  Thread-safe as far as the set-up goes (a mutex guards the
 * per-device table); the sharing rule above still applies. */
int nb_gravity_accel_static(int64_t n, const float* posm, float G, float eps, float* acc, void* cuda_stream,
                            int* cuda_error);
int64_t nb_gravity_accel_static_max_n(void);

void nb_destroy(nb_ctx* ctx);
const char* nb_strerror(int status);
int nb_last_cuda_error(nb_ctx* ctx);

/* Host-only scalars (no ctx).
 * Eq. 3: Roche-lobe radius / separation of the star whose mass is
 * the numerator of mass_ratio; k is the constant printed as 0.69 (standard 0.6, A9).
 * nb_l1_distance: distance of L1 from the primary in units of the separation,
 * q = m2/m1.  NaN on invalid arguments. */
double nb_roche_lobe_radius(double mass_ratio, double k);
double nb_l1_distance(double q);

#ifdef __cplusplus
}
#endif
#endif /* NB_H_ */
