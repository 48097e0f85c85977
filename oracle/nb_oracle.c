/*
 * oracle/nb_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision CPU restatement of what the hot path of
 * arXiv 2303.12166 computes: the all-pairs element-element acceleration
 * (Eqs. 4-6), the leapfrog step that consumes it
 * (PAPER.md:89), the expanding-star rule, and the two host
 * scalars the configs need (Roche-lobe radius, Eq. 3; the L1
 * point).  It is the *definition* written out: one i loop, one
 * j loop, no blocking, no fusion, no reordering.  OpenMP splits the i loop
 * only; every a_i is summed in j order, so results are bit-identical for any
 * thread count.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant with the CUDA library in paper_2303_12166_b200/csrc and neither
 * includes the other.
 *
 * Readings of the paper:
 *   A1  last term of the repulsion bracket is r^3/12 (lens_mode 0); the literal
 *       printed r^2/12 is lens_mode 1.
 *   A2  cross-star pair: R_ij = (R_i + R_j)/2, in contact iff r < R_i + R_j.
 *   A3  j != i only; a coincident pair (r == 0) contributes nothing.
 *   A4  a_i = (1/m_i) sum_j F_ij * unit(i->j), positive F attractive.
 *   A5  converging iff rdot < -v_dead; everything else takes gamma*beta.
 *   A6  pairs with |rdot + v_dead| <= tau_s are reported in delta_i (either
 *       branch is acceptable for a comparison in another precision).
 *   A7  kick-drift-kick with the end-of-step acceleration cached; a(x_{n+1})
 *       sees the half-step velocity.
 *   A8  R_s(n) linear in the step count n, then rounded to float (the model
 *       parameter is single precision, like the state).
 *   A12 U_rep(r) = gamma*pi*(R^4 - 4/3 R^3 r + 1/2 R^2 r^2 - r^4/48), with gamma.
 *
 * Pins: tests/test_oracle_*.py (-m "not gpu").  Unpinned by the paper: the
 * values of gamma, beta and the rdot == 0 tie (parity unpinned; fixed only by
 * the A5/A13 conventions).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

typedef struct {
    double G;        /* Eq. 4 */
    double eps;      /* Eq. 4 softening, (r + eps)^2 */
    double gamma;    /* Eq. 5 repulsion strength; 0 disables contact terms */
    double beta;     /* Eq. 6 reduction fraction */
    double v_dead;   /* A5 */
    double tau_s;    /* A6 */
    int32_t lens_mode; /* A1: 0 -> r^3/12, 1 -> r^2/12 as printed */
    int32_t pad_;
} orc_params;

/* pi * (4/3 R^3 - R^2 r + r^{3|2}/12): the bracket of Eqs. 5/6
 * times pi, in the expanded form the paper prints. */
double orc_lens_volume(double r, double R, int32_t lens_mode)
{
    double last = (lens_mode == 0) ? r * r * r : r * r;
    return M_PI * (4.0 / 3.0 * R * R * R - R * R * r + last / 12.0);
}

/* A12: U_rep(r) = integral_r^{2R} gamma*pi*V(r') dr' (lens_mode 0 only). */
double orc_rep_potential(double r, double R, double gamma)
{
    return gamma * M_PI * (R * R * R * R - 4.0 / 3.0 * R * R * R * r
                           + 0.5 * R * R * r * r - r * r * r * r / 48.0);
}

/*
 * Accelerations of the elements listed in rows[0..nrows) (rows == NULL: all n,
 * nrows ignored) from all n elements.  x, v: [n][3]; m, star: [n]; R[2]: element
 * radius per star.  Outputs (any may be NULL except a): a [nrows][3];
 * kappa[nrows] = sum_j |a_ij| / |a_i| (conditioning, for diagnosis);
 * delta[nrows] = sum over A6-ambiguous contact pairs of (1-beta)*gamma*pi*V/m_i.
 */
void orc_accel(int64_t n, const double *x, const double *v, const double *m,
               const int32_t *star, const double *R, const orc_params *p,
               int64_t nrows, const int64_t *rows,
               double *a, double *kappa, double *delta)
{
    const int64_t nr = rows ? nrows : n;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < nr; ++k) {
        const int64_t i = rows ? rows[k] : k;
        double ax = 0.0, ay = 0.0, az = 0.0, sabs = 0.0, dl = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;                                   /* A3 */
            const double dx = x[3 * j + 0] - x[3 * i + 0];
            const double dy = x[3 * j + 1] - x[3 * i + 1];
            const double dz = x[3 * j + 2] - x[3 * i + 2];
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            if (r == 0.0) continue;                                 /* A3 */
            double f = p->G * m[j] / ((r + p->eps) * (r + p->eps)); /* Eq. 4 / m_i */
            const double Rij = 0.5 * (R[star[i]] + R[star[j]]);     /* A2 */
            if (p->gamma > 0.0 && r < 2.0 * Rij) {                  /* in contact */
                const double V = orc_lens_volume(r, Rij, p->lens_mode);
                const double rdot = (dx * (v[3 * j + 0] - v[3 * i + 0])
                                   + dy * (v[3 * j + 1] - v[3 * i + 1])
                                   + dz * (v[3 * j + 2] - v[3 * i + 2])) / r;
                const double g = (rdot < -p->v_dead) ? p->gamma            /* Eq. 5 */
                                                     : p->gamma * p->beta; /* Eq. 6 */
                f -= g * V / m[i];
                if (fabs(rdot + p->v_dead) <= p->tau_s)             /* A6 */
                    dl += (1.0 - p->beta) * p->gamma * fabs(V) / m[i];
            }
            ax += f * dx / r;
            ay += f * dy / r;
            az += f * dz / r;
            sabs += fabs(f);
        }
        a[3 * k + 0] = ax; a[3 * k + 1] = ay; a[3 * k + 2] = az;
        if (kappa) {
            const double an = sqrt(ax * ax + ay * ay + az * az);
            kappa[k] = an > 0.0 ? sabs / an : INFINITY;
        }
        if (delta) delta[k] = dl;
    }
}

/*
 * The contact pairs of the elements listed in rows[0..nrows) (rows == NULL: all n): every j != i
 * with 0 < r < R_i + R_j ("in contact"; A2, A3), in j order.  count[k] receives the
 * number of such pairs of row k; the first min(count[k], cap) of them are written to
 * jj / rr / rd [k*cap + ...] as (j, r, rdot = d.(v_j - v_i)/r) -- the quantity whose sign selects
 * Eq. 5 or Eq. 6 (A5).  No force arithmetic here: the tests use the list to derive,
 * from the distribution of rdot, how many pairs can sit within tau_s of the switch (A6), and as a
 * brute-force count of the contacts a spatial search must find.
 */
void orc_contact_list(int64_t n, const double *x, const double *v, const int32_t *star,
                      const double *R, int64_t nrows, const int64_t *rows, int64_t cap,
                      int64_t *count, int64_t *jj, double *rr, double *rd)
{
    const int64_t nr = rows ? nrows : n;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < nr; ++k) {
        const int64_t i = rows ? rows[k] : k;
        int64_t c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const double dx = x[3 * j + 0] - x[3 * i + 0];
            const double dy = x[3 * j + 1] - x[3 * i + 1];
            const double dz = x[3 * j + 2] - x[3 * i + 2];
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            if (r == 0.0 || !(r < R[star[i]] + R[star[j]])) continue;
            if (c < cap) {
                jj[k * cap + c] = j;
                rr[k * cap + c] = r;
                rd[k * cap + c] = (dx * (v[3 * j + 0] - v[3 * i + 0])
                                 + dy * (v[3 * j + 1] - v[3 * i + 1])
                                 + dz * (v[3 * j + 2] - v[3 * i + 2])) / r;
            }
            ++c;
        }
        count[k] = c;
    }
}

/* Expanding-star rule (A8): element radius of each star at step n. */
void orc_radii(int64_t nstep, const double *R_start, const double *R_end,
               int64_t n_ramp, double *R)
{
    for (int s = 0; s < 2; ++s) {
        double Rs = R_start[s];
        if (n_ramp > 0) {
            const int64_t nn = nstep < n_ramp ? nstep : n_ramp;
            Rs = R_start[s] + (R_end[s] - R_start[s]) * (double)nn / (double)n_ramp;
        }
        R[s] = (double)(float)Rs;   /* the model parameter is single precision */
    }
}

/*
 * k kick-drift-kick leapfrog steps (A7) starting at step count n0.
 * x, v updated in place.  acc [n][3]: on entry the cached a(x_n0) if
 * *have_acc != 0, otherwise it is computed first; on exit a(x_{n0+k}).
 */
void orc_step(int64_t n, double *x, double *v, const double *m,
              const int32_t *star, const orc_params *p,
              const double *R_start, const double *R_end, int64_t n_ramp,
              double dt, int64_t n0, int64_t k, double *acc, int32_t *have_acc)
{
    double R[2];
    if (!*have_acc) {
        orc_radii(n0, R_start, R_end, n_ramp, R);
        orc_accel(n, x, v, m, star, R, p, 0, NULL, acc, NULL, NULL);
        *have_acc = 1;
    }
    for (int64_t s = 0; s < k; ++s) {
        for (int64_t i = 0; i < 3 * n; ++i) v[i] += 0.5 * dt * acc[i];
        for (int64_t i = 0; i < 3 * n; ++i) x[i] += dt * v[i];
        orc_radii(n0 + s + 1, R_start, R_end, n_ramp, R);
        orc_accel(n, x, v, m, star, R, p, 0, NULL, acc, NULL, NULL);
        for (int64_t i = 0; i < 3 * n; ++i) v[i] += 0.5 * dt * acc[i];
    }
}

/*
 * out[0..10]: KE, U_grav, U_rep, E, Px, Py, Pz, Lx, Ly, Lz, |sum m_i a_i|
 * (the last only if acc != NULL, else 0).  U_grav = -sum_{i<j} G m_i m_j/(r+eps)
 * (the potential whose gradient is Eq. 4); U_rep per A12 (lens_mode 0).
 */
void orc_energy(int64_t n, const double *x, const double *v, const double *m,
                const int32_t *star, const double *R, const orc_params *p,
                const double *acc, double *out)
{
    double ke = 0, ug = 0, ur = 0, P[3] = {0, 0, 0}, L[3] = {0, 0, 0}, F[3] = {0, 0, 0};
    for (int64_t i = 0; i < n; ++i) {
        const double *xi = x + 3 * i, *vi = v + 3 * i;
        ke += 0.5 * m[i] * (vi[0] * vi[0] + vi[1] * vi[1] + vi[2] * vi[2]);
        for (int c = 0; c < 3; ++c) P[c] += m[i] * vi[c];
        L[0] += m[i] * (xi[1] * vi[2] - xi[2] * vi[1]);
        L[1] += m[i] * (xi[2] * vi[0] - xi[0] * vi[2]);
        L[2] += m[i] * (xi[0] * vi[1] - xi[1] * vi[0]);
        if (acc) for (int c = 0; c < 3; ++c) F[c] += m[i] * acc[3 * i + c];
    }
#pragma omp parallel for schedule(dynamic, 64) reduction(+ : ug, ur)
    for (int64_t i = 0; i < n; ++i) {
        for (int64_t j = i + 1; j < n; ++j) {
            const double dx = x[3 * j + 0] - x[3 * i + 0];
            const double dy = x[3 * j + 1] - x[3 * i + 1];
            const double dz = x[3 * j + 2] - x[3 * i + 2];
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            ug -= p->G * m[i] * m[j] / (r + p->eps);
            const double Rij = 0.5 * (R[star[i]] + R[star[j]]);
            if (p->gamma > 0.0 && r < 2.0 * Rij)
                ur += orc_rep_potential(r, Rij, p->gamma);
        }
    }
    out[0] = ke; out[1] = ug; out[2] = ur; out[3] = ke + ug + ur;
    for (int c = 0; c < 3; ++c) { out[4 + c] = P[c]; out[7 + c] = L[c]; }
    out[10] = sqrt(F[0] * F[0] + F[1] * F[1] + F[2] * F[2]);
}

/* Eq. 3: Roche-lobe radius in units of the separation, for the
 * star whose mass is the numerator of `mass_ratio` (A11).  k is the constant
 * the paper prints as 0.69 (A9; the standard value is 0.6). */
double orc_roche_lobe_radius(double mass_ratio, double k)
{
    const double q23 = pow(mass_ratio, 2.0 / 3.0);
    const double q13 = pow(mass_ratio, 1.0 / 3.0);
    return 0.49 * q23 / (k * q23 + log(1.0 + q13));
}

/* Distance of L1 from the primary m1, in units of the separation, for
 * q = m2/m1.  Force balance on the line of centres in the
 * co-rotating frame with G(m1+m2) = a = 1, so omega = 1: gravity of both
 * masses plus the centrifugal term vanish; solved by bisection. */
double orc_l1_distance(double q)
{
    const double mu1 = 1.0 / (1.0 + q), mu2 = q / (1.0 + q);
    const double x1 = -q / (1.0 + q), x2 = 1.0 / (1.0 + q);
    double lo = x1 + 1e-12, hi = x2 - 1e-12;
    for (int it = 0; it < 200; ++it) {
        const double xm = 0.5 * (lo + hi);
        const double f = -mu1 / ((xm - x1) * (xm - x1)) + mu2 / ((x2 - xm) * (x2 - xm)) + xm;
        if (f < 0.0) lo = xm; else hi = xm;   /* f increases monotonically on (x1,x2) */
    }
    return 0.5 * (lo + hi) - x1;
}
