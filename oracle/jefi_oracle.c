/*
 * jefi_oracle.c -- fp64 CPU oracle for the discretised Jefimenko sums.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call this.  It shares no code,
 * header, table or helper with the CUDA path (paper_2104_05426_b200/csrc, include/jefi.h)
 * and includes nothing but libc.  It is the plain definition written out: a triple loop
 * over source cells per observation point, in the paper's order, with no blocking,
 * fusion, pre-scaling or reordering, so that it can be checked against the paper by eye.
 *
 * What it computes (Sec. 2.2 Eq. (4)-(6)), per observation point r and
 * evaluation step n (t = t0 + n*dt):
 *
 *   E(r,t) = dV/(4 pi) * sum_{i,j,k} [ d*( rho/R^3 + rho_dot/(c R^2) ) - J_dot/(c^2 R) ]
 *   B(r,t) = dV/(4 pi) * sum_{i,j,k} [ ( J/R^3 + J_dot/(c R^2) ) x d ]
 *
 *   d = r - r'_{ijk},  R = |d|,  all source quantities taken at the retarded step
 *   m = n - floor(R/(c dt) + 0.5)                       (Eq. (6); reading Q3)
 *
 * Readings of the paper (listed in DESIGN.md):
 *   Q1  sign of the J_dot/R term: MINUS, as in Eq. (4), not the '+' of Eq. (1).
 *   Q2  time derivative: deriv_mode 0 = centred difference inside the stored history,
 *       one-sided at m=0 and m=T-1 (north_star); deriv_mode 1 = the paper's backward
 *       difference (f(t_r)-f(t_r-dt))/dt with f[-1] = 0.
 *   Q3  nearest stored step on the delay: k = floor(R/(c dt) + 0.5).
 *   Q4  m < 0 (before the first stored step) contributes zero (Eq. (7),(9)).
 *   Q5  coarse screening: skip the cell iff R < 0.5*min(dx,dy,dz), strict.
 *   Q6  r'_{ijk} = origin + (i,j,k)*spacing are cell centres.
 *   Q7  explicit c with the weights d/R^3, d/(c R^2), 1/(c^2 R), and no extra power of c on B.
 *   Q8  B ~ +(J x d)  ==  the paper's -(d x J).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): hand-summed worked example, Coulomb,
 * Biot-Savart (exact hand sum and closed form), linearity, switch-on causality with its
 * closed-form precursor, time translation, late-time constancy, c-rescaling invariance,
 * far-zone radiation (fixes Q1 and Q8 together), mirror symmetry, and the paper's X1
 * legend magnitude.  Agreement with the *continuum* integral is "parity unpinned" beyond
 * the paper's own 3-14 %: the Mathematica results are not available.
 *
 * Layouts: rho[T][N_s], J[T][3][N_s], linear cell index j = (kz*ny + jy)*nx + ix (x fastest).
 * in_is_f32 != 0: the arrays hold float and are promoted element-wise to double, i.e. an
 * fp32 run's inputs are the fp32-rounded values and nothing else is rounded.
 * obs_xyz[n_obs][3] are explicit points; outputs E[3][n_obs], B[3][n_obs] (component planes).
 */
#include <math.h>
#include <pthread.h>
#include <stddef.h>
#include <stdlib.h>

typedef struct {
    int nx, ny, nz;
    double ox, oy, oz, hx, hy, hz;
    const void *rho, *J;
    int in_is_f32, T;
    double dt, c;
    int deriv_mode, n;
    long n_obs;
    const double *obs;
    double *E, *B;
    long begin, end;
} oracle_job;

/* value of a stored scalar field f[m][j] (m-th snapshot, cell j); zero before the history */
static double hist_at(const void *base, int is_f32, long plane_stride, long comp_off,
                      int m, long j)
{
    if (m < 0) return 0.0;
    size_t idx = (size_t)m * (size_t)plane_stride + (size_t)comp_off + (size_t)j;
    return is_f32 ? (double)((const float *)base)[idx] : ((const double *)base)[idx];
}

/* time derivative D(f, m, j) -- reading Q2 */
static double hist_ddt(const void *base, int is_f32, long plane_stride, long comp_off,
                       int m, long j, int T, double dt, int deriv_mode)
{
    if (deriv_mode == 1) {               /* paper, Eq. (4)-(5): backward, f[-1] = 0 */
        return (hist_at(base, is_f32, plane_stride, comp_off, m, j) -
                hist_at(base, is_f32, plane_stride, comp_off, m - 1, j)) / dt;
    }
    if (T == 1) return 0.0;
    if (m == 0)
        return (hist_at(base, is_f32, plane_stride, comp_off, 1, j) -
                hist_at(base, is_f32, plane_stride, comp_off, 0, j)) / dt;
    if (m == T - 1)
        return (hist_at(base, is_f32, plane_stride, comp_off, T - 1, j) -
                hist_at(base, is_f32, plane_stride, comp_off, T - 2, j)) / dt;
    return (hist_at(base, is_f32, plane_stride, comp_off, m + 1, j) -
            hist_at(base, is_f32, plane_stride, comp_off, m - 1, j)) / (2.0 * dt);
}

static void *oracle_worker(void *arg)
{
    const oracle_job *q = (const oracle_job *)arg;
    const long Ns = (long)q->nx * q->ny * q->nz;
    const double c = q->c, dt = q->dt;
    double hmin = q->hx;
    if (q->hy < hmin) hmin = q->hy;
    if (q->hz < hmin) hmin = q->hz;
    const double rcut = 0.5 * hmin;                         /* Q5 */
    const double dV = q->hx * q->hy * q->hz;                /* dOmega' */
    const double pi = 3.14159265358979323846;
    const double pref = dV / (4.0 * pi);

    for (long i = q->begin; i < q->end; ++i) {
        const double rx = q->obs[3 * i + 0], ry = q->obs[3 * i + 1], rz = q->obs[3 * i + 2];
        double Ex = 0, Ey = 0, Ez = 0, Bx = 0, By = 0, Bz = 0;
        for (int kz = 0; kz < q->nz; ++kz)
        for (int jy = 0; jy < q->ny; ++jy)
        for (int ix = 0; ix < q->nx; ++ix) {
            const long j = ((long)kz * q->ny + jy) * q->nx + ix;
            const double sx = q->ox + ix * q->hx;           /* Q6: cell centre */
            const double sy = q->oy + jy * q->hy;
            const double sz = q->oz + kz * q->hz;
            const double dx = rx - sx, dy = ry - sy, dz = rz - sz;
            const double R = sqrt(dx * dx + dy * dy + dz * dz);
            if (R < rcut) continue;                         /* Q5: strict '<' */
            const long k = (long)floor(R / (c * dt) + 0.5); /* Q3 */
            const long ml = (long)q->n - k;
            if (ml < 0) continue;                           /* Q4 */
            const int m = (int)ml;

            const double rho  = hist_at(q->rho, q->in_is_f32, Ns, 0, m, j);
            const double Jx   = hist_at(q->J, q->in_is_f32, 3 * Ns, 0 * Ns, m, j);
            const double Jy   = hist_at(q->J, q->in_is_f32, 3 * Ns, 1 * Ns, m, j);
            const double Jz   = hist_at(q->J, q->in_is_f32, 3 * Ns, 2 * Ns, m, j);
            const double rhod = hist_ddt(q->rho, q->in_is_f32, Ns, 0, m, j, q->T, dt, q->deriv_mode);
            const double Jxd  = hist_ddt(q->J, q->in_is_f32, 3 * Ns, 0 * Ns, m, j, q->T, dt, q->deriv_mode);
            const double Jyd  = hist_ddt(q->J, q->in_is_f32, 3 * Ns, 1 * Ns, m, j, q->T, dt, q->deriv_mode);
            const double Jzd  = hist_ddt(q->J, q->in_is_f32, 3 * Ns, 2 * Ns, m, j, q->T, dt, q->deriv_mode);

            const double R2 = R * R, R3 = R2 * R;
            /* E: Eq. (4) */
            const double s = rho / R3 + rhod / (c * R2);
            Ex += dx * s - Jxd / (c * c * R);
            Ey += dy * s - Jyd / (c * c * R);
            Ez += dz * s - Jzd / (c * c * R);
            /* B: Eq. (5);  -(d x u) = u x d  (Q8) */
            const double ux = Jx / R3 + Jxd / (c * R2);
            const double uy = Jy / R3 + Jyd / (c * R2);
            const double uz = Jz / R3 + Jzd / (c * R2);
            Bx += uy * dz - uz * dy;
            By += uz * dx - ux * dz;
            Bz += ux * dy - uy * dx;
        }
        q->E[0 * q->n_obs + i] = pref * Ex;
        q->E[1 * q->n_obs + i] = pref * Ey;
        q->E[2 * q->n_obs + i] = pref * Ez;
        q->B[0 * q->n_obs + i] = pref * Bx;
        q->B[1 * q->n_obs + i] = pref * By;
        q->B[2 * q->n_obs + i] = pref * Bz;
    }
    return NULL;
}

/* returns 0 on success, 1 on invalid arguments */
int jefi_oracle_fields(const int *n_src, const double *origin_src, const double *spacing_src,
                       const void *rho, const void *J, int in_is_f32, int T,
                       double dt, double c, int deriv_mode, int step_n,
                       long n_obs, const double *obs_xyz,
                       double *E_out, double *B_out, int nthreads)
{
    if (!n_src || !origin_src || !spacing_src || !rho || !J || !E_out || !B_out) return 1;
    if (n_obs > 0 && !obs_xyz) return 1;
    if (n_src[0] <= 0 || n_src[1] <= 0 || n_src[2] <= 0 || T <= 0) return 1;
    if (!(dt > 0) || !(c > 0) || step_n < 0 || step_n >= T) return 1;
    if (deriv_mode != 0 && deriv_mode != 1) return 1;
    if (nthreads < 1) nthreads = 1;
    if (nthreads > 256) nthreads = 256;
    if ((long)nthreads > n_obs) nthreads = n_obs > 0 ? (int)n_obs : 1;

    oracle_job jobs[256];
    pthread_t tid[256];
    const long per = (n_obs + nthreads - 1) / nthreads;
    for (int t = 0; t < nthreads; ++t) {
        oracle_job *q = &jobs[t];
        q->nx = n_src[0]; q->ny = n_src[1]; q->nz = n_src[2];
        q->ox = origin_src[0]; q->oy = origin_src[1]; q->oz = origin_src[2];
        q->hx = spacing_src[0]; q->hy = spacing_src[1]; q->hz = spacing_src[2];
        q->rho = rho; q->J = J; q->in_is_f32 = in_is_f32; q->T = T;
        q->dt = dt; q->c = c; q->deriv_mode = deriv_mode; q->n = step_n;
        q->n_obs = n_obs; q->obs = obs_xyz; q->E = E_out; q->B = B_out;
        q->begin = t * per;
        q->end = (t + 1) * per < n_obs ? (t + 1) * per : n_obs;
        if (q->begin > q->end) q->begin = q->end;
    }
    if (nthreads == 1) {
        oracle_worker(&jobs[0]);
        return 0;
    }
    for (int t = 0; t < nthreads; ++t) pthread_create(&tid[t], NULL, oracle_worker, &jobs[t]);
    for (int t = 0; t < nthreads; ++t) pthread_join(tid[t], NULL);
    return 0;
}

/* Retarded-step lag k = floor(R/(c dt) + 0.5) for explicit (obs point, source cell) pairs.
 * Used by tests that count GPU-vs-fp64 index mismatches (parity report). */
long jefi_oracle_lag(double rx, double ry, double rz, double sx, double sy, double sz,
                     double dt, double c)
{
    const double dx = rx - sx, dy = ry - sy, dz = rz - sz;
    const double R = sqrt(dx * dx + dy * dy + dz * dz);
    return (long)floor(R / (c * dt) + 0.5);
}
