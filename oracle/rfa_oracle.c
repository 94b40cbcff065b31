/*
 * rfa_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of the hot path of arXiv 1907.05709 (Kath, Handels, Mastmeyer):
 * explicit finite-difference time stepping of the simplified bioheat equation on a labelled voxel
 * volume.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA library
 * (paper_1907_05709_b200/csrc) and is deliberately written in a different algebraic form: Eq. 12
 * is evaluated un-factored, in SI units, voxel by voxel, exactly in the paper's order.
 *
 * Passages followed (line numbers of /root/reference/PAPER.md):
 *   Eq. 9   :102   rho c_p dT/dt = div(K grad T) + w_b c_b (T_a - T) + Q_m
 *   Eq. 11  :112   second difference (T_{i+1} - 2 T_i + T_{i-1}) / (dx)^2, per axis
 *   Eq. 12  :117   explicit Euler voxel update, parameters looked up voxel-wise (:120)
 *   Eq. 13  :122-125 + Alg. 1 :306,:313  vessel / needle-tip voxels keep their temperature
 *   Alg. 1  :296-319 one sweep over all voxels per time step
 *   Alg. 2  :321-337 two buffers, swapped after every step
 *   :37     total necrosis at temperatures "exceeding 60 C"  (read as T >= 60, sticky; R-11/R-12)
 *
 * Readings where the paper is silent or garbled are listed in DESIGN.md section 3 (R-1..R-26); the
 * ones that shape this file: K multiplies the SUM of the three quotients (R-1); spacing is given
 * in millimetres and converted to metres (R-2); the centre voxel's K times the plain 7-point
 * Laplacian (R-3); held voxels are Dirichlet (R-4); outer grid faces are zero-flux by replication,
 * missing neighbour := the voxel itself (R-7); constant-power voxels add Q inside the bracket (R-17).
 *
 * Pins (tests/test_oracle_pins.py): exact DCT closed form on anisotropic non-cubic grids, uniform
 * relaxation to T_a + Q_m/beta, dense-matrix brute force on 4^3 and 6x5x4, weighted-energy
 * invariant, checkerboard stability bound, monotone heating, max principle, 48-fold symmetry,
 * Green's function refinement (Eq. 2), erfc plane source (Eq. 4 with constant h), linear steady
 * state (Fig. 2b), tridiagonal steady state with perfusion.  The paper prints no temperature value
 * anywhere (all results are figures), so parity with the paper's own curves is UNPINNED.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* One time step (one iteration of the while-loop of Alg. 1).
 *   lab[v]    label id of voxel v, indexes the per-label constant arrays ("voxel-wise")
 *   held[v]   nonzero: vessel / fixed label / Dirichlet needle voxel -> copied (Alg. 1 :313)
 *   power[v]  nonzero: constant power source Q [W/m^3] added to the bracket of Eq. 12 (R-17)
 *   T -> Tn   temperature images in deg C; necro[v] |= (Tn[v] >= t_necro)  (sticky, R-12)
 * Memory order: x fastest, idx = i + nx*(j + ny*k)  (R-23).  dx, dy, dz in METRES.
 */
void rfa_oracle_step(int nx, int ny, int nz, double dx, double dy, double dz,
                     const uint8_t *lab, const uint8_t *held, const uint8_t *power,
                     const double *K, const double *rho, const double *cp,
                     const double *wb_cb, const double *q_m,
                     double t_a, double q_power, double dt, double t_necro,
                     const double *T, double *Tn, uint8_t *necro)
{
    int k;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (k = 0; k < nz; ++k) {
        int km = k > 0 ? k - 1 : 0;               /* zero flux: missing neighbour = the voxel itself */
        int kp = k < nz - 1 ? k + 1 : nz - 1;
        for (int j = 0; j < ny; ++j) {
            int jm = j > 0 ? j - 1 : 0;
            int jp = j < ny - 1 ? j + 1 : ny - 1;
            for (int i = 0; i < nx; ++i) {
                int im = i > 0 ? i - 1 : 0;
                int ip = i < nx - 1 ? i + 1 : nx - 1;
                size_t v = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                double t = T[v];
                double tn;
                if (held[v]) {
                    tn = t;                                              /* Eq. 13 / Alg. 1 :313 */
                } else {
                    double xm = T[(size_t)im + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k)];
                    double xp = T[(size_t)ip + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k)];
                    double ym = T[(size_t)i + (size_t)nx * ((size_t)jm + (size_t)ny * (size_t)k)];
                    double yp = T[(size_t)i + (size_t)nx * ((size_t)jp + (size_t)ny * (size_t)k)];
                    double zm = T[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)km)];
                    double zp = T[(size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)kp)];
                    int l = lab[v];
                    /* Eq. 11, one quotient per axis */
                    double d2x = (xm - 2.0 * t + xp) / (dx * dx);
                    double d2y = (ym - 2.0 * t + yp) / (dy * dy);
                    double d2z = (zm - 2.0 * t + zp) / (dz * dz);
                    /* right-hand side of Eq. 12: K*(sum) + w_b c_b (T_a - T) + Q_m  (+ Q, R-17) */
                    double rhs = K[l] * (d2x + d2y + d2z) + wb_cb[l] * (t_a - t) + q_m[l];
                    if (power[v]) rhs += q_power;
                    tn = t + dt / (rho[l] * cp[l]) * rhs;
                }
                Tn[v] = tn;
                if (tn >= t_necro) necro[v] = 1;
            }
        }
    }
}

/* One time step with CONSERVATIVE heterogeneous conduction (R-28):
 * Eq. 9 writes div(K grad T) before Eq. 10/12 pull a constant K out of the divergence.
 * Finite-volume form on the voxel grid: the heat flux through the face between voxel c and its face
 * neighbour n is  Kf (T_n - T_c) / h  with the harmonic mean  Kf = 2 K_c K_n / (K_c + K_n)  of the two
 * voxels' conductivities (two slabs of thickness h/2 in series), so
 *   T_c' = T_c + dt/(rho c_p) * [ sum over the 6 faces Kf (T_n - T_c) / h_axis^2
 *                                 + w_b c_b (T_a - T_c) + Q_m (+ Q) ]
 * Outer grid faces carry no flux (the missing neighbour is the voxel itself, R-7).  Held voxels are
 * copied and act on their neighbours through the face term with their own label's K.
 * Arguments as rfa_oracle_step. */
void rfa_oracle_step_cons(int nx, int ny, int nz, double dx, double dy, double dz,
                          const uint8_t *lab, const uint8_t *held, const uint8_t *power,
                          const double *K, const double *rho, const double *cp,
                          const double *wb_cb, const double *q_m,
                          double t_a, double q_power, double dt, double t_necro,
                          const double *T, double *Tn, uint8_t *necro)
{
    int k;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (k = 0; k < nz; ++k) {
        for (int j = 0; j < ny; ++j) {
            for (int i = 0; i < nx; ++i) {
                size_t v = (size_t)i + (size_t)nx * ((size_t)j + (size_t)ny * (size_t)k);
                double t = T[v];
                double tn;
                if (held[v]) {
                    tn = t;
                } else {
                    int l = lab[v];
                    double kc = K[l];
                    double flux = 0.0;                     /* sum of Kf (T_n - T_c) / h^2 over the faces */
                    for (int f = 0; f < 6; ++f) {
                        int ii = i, jj = j, kk = k;
                        double h;
                        if (f == 0) { ii = i - 1; h = dx; }
                        else if (f == 1) { ii = i + 1; h = dx; }
                        else if (f == 2) { jj = j - 1; h = dy; }
                        else if (f == 3) { jj = j + 1; h = dy; }
                        else if (f == 4) { kk = k - 1; h = dz; }
                        else { kk = k + 1; h = dz; }
                        if (ii < 0 || ii >= nx || jj < 0 || jj >= ny || kk < 0 || kk >= nz) continue;   /* no flux */
                        size_t n = (size_t)ii + (size_t)nx * ((size_t)jj + (size_t)ny * (size_t)kk);
                        double kn = K[lab[n]];
                        double kf = 2.0 * kc * kn / (kc + kn);
                        flux += kf * (T[n] - t) / (h * h);
                    }
                    double rhs = flux + wb_cb[l] * (t_a - t) + q_m[l];
                    if (power[v]) rhs += q_power;
                    tn = t + dt / (rho[l] * cp[l]) * rhs;
                }
                Tn[v] = tn;
                if (tn >= t_necro) necro[v] = 1;
            }
        }
    }
}

/* nsteps iterations with the two buffers of Alg. 2.  On return the current
 * temperature image is in T (buf is scratch of the same size).  conservative != 0 selects
 * rfa_oracle_step_cons (row f1), 0 the paper's Eq. 12 as printed. */
void rfa_oracle_run(int nx, int ny, int nz, double dx, double dy, double dz,
                    const uint8_t *lab, const uint8_t *held, const uint8_t *power,
                    const double *K, const double *rho, const double *cp,
                    const double *wb_cb, const double *q_m,
                    double t_a, double q_power, double dt, double t_necro,
                    int nsteps, double *T, double *buf, uint8_t *necro, int conservative)
{
    double *a = T, *b = buf;
    for (int n = 0; n < nsteps; ++n) {
        if (conservative)
            rfa_oracle_step_cons(nx, ny, nz, dx, dy, dz, lab, held, power, K, rho, cp, wb_cb, q_m,
                                 t_a, q_power, dt, t_necro, a, b, necro);
        else
            rfa_oracle_step(nx, ny, nz, dx, dy, dz, lab, held, power, K, rho, cp, wb_cb, q_m,
                            t_a, q_power, dt, t_necro, a, b, necro);
        double *t = a; a = b; b = t;
    }
    if (a != T) memcpy(T, a, sizeof(double) * (size_t)nx * (size_t)ny * (size_t)nz);
}

int rfa_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void rfa_oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
