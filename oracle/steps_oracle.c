/*
 * steps_oracle.c -- CPU oracle for the StePS hot path (arXiv:1811.05903).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or constant with paper_1811_05903_b200/csrc (the CUDA
 * path) and neither side includes the other.
 *
 * It is the plain definition written out: every ordered pair (i, j != i) goes through
 * the paper's spline pair law with pair softening h_i + h_j, in fp64, in the paper's
 * notation, with no tiling, no symmetry trick, no far/near split, no reciprocal-sqrt
 * tricks.  The only liberty is the summation: each component is accumulated with
 * Neumaier's compensated sum so that the oracle's own summation error (~1e-16
 * relative, independent of order) is far below the 1e-12 parity bar the CUDA fp64
 * path is held to.  OpenMP over i only.
 *
 * Citations are PAPER.md line numbers (L..) and equation numbers; "reading #k" refers
 * to the numbered readings in DESIGN.md (taken from SURVEY.md 8(c.4)).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): hand values of Eq. 4, branch
 * continuity, the two-body closed form, exact Newtonian r >= h, shell theorem on
 * regular polyhedra and a Fibonacci shell, Newton's third law, symmetries, an
 * independent numpy longdouble brute force on N <= 8, RK4 a(t) vs closed forms, drag
 * and background-term closed forms with 2nd-order convergence, Kepler orbit; Eq. 12 time step against the two-body
 * closed form, its scaling laws, the dt_max clamp and a numpy brute force; the momentum diagnostic against hand-typed
 * three-particle values and a numpy longdouble brute force; the growth rate (oracle/steps_oracle.py, config-4 initial
 * velocities) against the hypergeometric closed form of flat LCDM.
 * Parity status: every function below is pinned (none "parity unpinned"); the choice
 * of how the drag enters the kick (reading #8) is a reading the paper does not fix.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ pair law */

/* PAPER.md Eq. 4 (L57-61): the spline-softened 1/r^2.  Reading #1: the three branches
 * as printed (the "- \\ -48 r^2/h^4" is a line-break artefact, one minus sign).
 * Reading #2: r < h/2 | h/2 <= r < h | r >= h (the function is continuous). */
double oracle_spline_F(double r, double h)
{
    if (r < 0.5 * h) {
        return 32.0 * r * r * r * r / pow(h, 6) - 38.4 * r * r * r / pow(h, 5) + 32.0 * r / (3.0 * h * h * h);
    } else if (r < h) {
        return -32.0 * r * r * r * r / (3.0 * pow(h, 6)) + 38.4 * r * r * r / pow(h, 5)
               - 48.0 * r * r / pow(h, 4) + 64.0 * r / (3.0 * h * h * h) - 1.0 / (15.0 * r * r);
    }
    return 1.0 / (r * r);
}

/* Neumaier compensated accumulation: (s, c) <- (s, c) + t. */
static inline void neumaier_add(double *s, double *c, double t)
{
    double u = *s + t;
    if (fabs(*s) >= fabs(t)) *c += (*s - u) + t;
    else                     *c += (t - u) + *s;
    *s = u;
}

/* ------------------------------------------------------------------ force sum */

/* PAPER.md Eq. 8 (L88), first term, with G = 1 and without the a^-3 (both enter through
 * the kick):   acc_i = sum_{j != i} m_j F(x_i - x_j, h_i + h_j),
 * F(x, h) = -calF(|x|, h) x/|x|   (Eq. 3).   Reading #3: the spline's h is the SUM
 * h_i + h_j.  Reading #4: j = i is skipped; a coincident distinct pair (r = 0) adds 0.
 *
 * pos: SoA [x | y | z], 3N doubles.  idx: n_idx particle indices to evaluate (NULL = all
 * N, n_idx ignored).  acc: SoA [ax | ay | az] over the evaluated particles (3 * count).
 * reverse_j != 0 runs the j loop backwards (used only to show order independence). */
void oracle_forces(const double *pos, const double *mass, const double *soft, long long N,
                   const long long *idx, long long n_idx, double *acc, int reverse_j)
{
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    const long long count = idx ? n_idx : N;
#pragma omp parallel for schedule(dynamic, 16)
    for (long long k = 0; k < count; ++k) {
        const long long i = idx ? idx[k] : k;
        double sx = 0, sy = 0, sz = 0, cx = 0, cy = 0, cz = 0;
        for (long long jj = 0; jj < N; ++jj) {
            const long long j = reverse_j ? N - 1 - jj : jj;
            if (j == i) continue;
            const double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];   /* x_i - x_j */
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            if (r == 0.0) continue;                                               /* reading #4 */
            const double h = soft[i] + soft[j];
            const double f = -mass[j] * oracle_spline_F(r, h);                    /* Eq. 3, G = 1 */
            neumaier_add(&sx, &cx, f * (dx / r));
            neumaier_add(&sy, &cy, f * (dy / r));
            neumaier_add(&sz, &cz, f * (dz / r));
        }
        acc[k] = sx + cx;
        acc[count + k] = sy + cy;
        acc[2 * count + k] = sz + cz;
    }
}

/* Quasi-periodic boundary conditions, Eq. 5 (L65-70): "only the leading term of the sum in Eq. 5 is kept
 * for each pair of particles", i.e. of all images x - nL of the separation vector the one of smallest length, in a cubic
 * box of side L.  Reading (#16): the leading term is taken component by component, n_c = round-half-even of
 * (x_c / L) (nearbyint under the default rounding mode), so a component of exactly L/2 keeps its sign; otherwise as
 * oracle_forces above (pair softening h_i + h_j, j = i skipped, r = 0 adds 0, G = 1, compensated sums). */
void oracle_forces_quasi_periodic(const double *pos, const double *mass, const double *soft, long long N, double L,
                                  const long long *idx, long long n_idx, double *acc)
{
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    const long long count = idx ? n_idx : N;               /* idx: the particles to evaluate, as in oracle_forces */
#pragma omp parallel for schedule(dynamic, 16)
    for (long long k = 0; k < count; ++k) {
        const long long i = idx ? idx[k] : k;
        double sx = 0, sy = 0, sz = 0, cx = 0, cy = 0, cz = 0;
        for (long long j = 0; j < N; ++j) {
            if (j == i) continue;
            double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];          /* x_i - x_j */
            dx -= L * nearbyint(dx / L);                                          /* leading image, Eq. 5 */
            dy -= L * nearbyint(dy / L);
            dz -= L * nearbyint(dz / L);
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            if (r == 0.0) continue;
            const double h = soft[i] + soft[j];
            const double f = -mass[j] * oracle_spline_F(r, h);
            neumaier_add(&sx, &cx, f * (dx / r));
            neumaier_add(&sy, &cy, f * (dy / r));
            neumaier_add(&sz, &cz, f * (dz / r));
        }
        acc[k] = sx + cx;
        acc[count + k] = sy + cy;
        acc[2 * count + k] = sz + cz;
    }
}

/* Periodic boundary conditions, Eq. 5 (L65-70) with the paper's cut: F(x, h) = sum over integer triplets n of
 * -G calF(|x - nL|, h) (x - nL)/|x - nL|, "the only valid triplets are where |x - nL| < 2.6 L is fulfilled".
 * Reading (#17): x is the separation x_i - x_j as it is (no prior wrapping: the set {x - nL} is the same for
 * every representative of x modulo L, so the sum does not depend on it); the triplets are searched in |n_c| <= 4 around
 * the nearest image, which contains every n with |x - nL| < 2.6 L; strict inequality as printed; the pair law with pair
 * softening h_i + h_j is applied to every image.  Plain loops, compensated sums. */
void oracle_forces_periodic_images(const double *pos, const double *mass, const double *soft, long long N, double L,
                                   const long long *idx, long long n_idx, double *acc)
{
    const double *x = pos, *y = pos + N, *z = pos + 2 * N;
    const double cut = 2.6 * L;
    const long long count = idx ? n_idx : N;               /* idx: the particles to evaluate, as in oracle_forces */
#pragma omp parallel for schedule(dynamic, 4)
    for (long long k = 0; k < count; ++k) {
        const long long i = idx ? idx[k] : k;
        double sx = 0, sy = 0, sz = 0, cx = 0, cy = 0, cz = 0;
        for (long long j = 0; j < N; ++j) {
            if (j == i) continue;
            const double h = soft[i] + soft[j];
            const double bx = x[i] - x[j], by = y[i] - y[j], bz = z[i] - z[j];
            const double ox = nearbyint(bx / L), oy = nearbyint(by / L), oz = nearbyint(bz / L);
            for (int n1 = -4; n1 <= 4; ++n1)
                for (int n2 = -4; n2 <= 4; ++n2)
                    for (int n3 = -4; n3 <= 4; ++n3) {
                        const double dx = bx - (ox + n1) * L, dy = by - (oy + n2) * L, dz = bz - (oz + n3) * L;
                        const double r = sqrt(dx * dx + dy * dy + dz * dz);
                        if (!(r < cut) || r == 0.0) continue;
                        const double f = -mass[j] * oracle_spline_F(r, h);
                        neumaier_add(&sx, &cx, f * (dx / r));
                        neumaier_add(&sy, &cy, f * (dy / r));
                        neumaier_add(&sz, &cz, f * (dz / r));
                    }
        }
        acc[k] = sx + cx;
        acc[count + k] = sy + cy;
        acc[2 * count + k] = sz + cz;
    }
}

/* ------------------------------------------------------------------ background */

typedef struct {
    double H0, Omega_m, Omega_r, Omega_L, Omega_k;
} oracle_cosmo;

/* PAPER.md Eq. 1 (L37):  H(a) = H0 sqrt(Om a^-3 + Or a^-4 + OL + Ok a^-2). */
double oracle_hubble(double a, const oracle_cosmo *c)
{
    return c->H0 * sqrt(c->Omega_m / (a * a * a) + c->Omega_r / (a * a * a * a) + c->Omega_L + c->Omega_k / (a * a));
}

/* a(t) advanced by classical 4th-order Runge-Kutta on da/dt = a H(a),
 * with the same step the N-body integrator uses. */
double oracle_rk4_scale_factor(double a, double dt, const oracle_cosmo *c)
{
    const double k1 = a * oracle_hubble(a, c);
    const double a2 = a + 0.5 * dt * k1;
    const double k2 = a2 * oracle_hubble(a2, c);
    const double a3 = a + 0.5 * dt * k2;
    const double k3 = a3 * oracle_hubble(a3, c);
    const double a4 = a + dt * k3;
    const double k4 = a4 * oracle_hubble(a4, c);
    return a + dt * (k1 + 2.0 * k2 + 2.0 * k3 + k4) / 6.0;
}

/* ------------------------------------------------------------------ KDK step */

/* One kick-drift-kick step, Eq. 9-11 (L98-109) applied to Eq. 8 (L88):
 *   x'' = a^-3 [ G sum_j m_j F + (4 pi G/3) rho_bar x ] - 2 H x'          (reading #6)
 * State in: x_n, v_n, acc_n = force sum at x_n (G = 1 units), *a = a_n.
 *   K(dt/2), explicit in the drag at (a_n, H_n)                          (reading #8)
 *   D(dt)
 *   a_{n+1} by RK4 (L127), H_{n+1} from Eq. 1                            (reading #9)
 *   one force evaluation at x_{n+1} (L96)
 *   K(dt/2), implicit in the drag at (a_{n+1}, H_{n+1})                  (reading #8)
 * B = (4 pi/3) rho_bar in G = 1 units; the acceleration used by the kicks is
 * G a^-3 (acc + B x).  With H0 = 0 and *a = 1 this is the static Newtonian mode (L92).
 * State out: x_{n+1}, v_{n+1}, acc_{n+1}, *a = a_{n+1}. */
void oracle_kdk_step(double *pos, double *vel, double *acc, const double *mass, const double *soft,
                     long long N, double *a, double dt, double G, double B, const oracle_cosmo *c)
{
    const long long M = 3 * N;
    const double a_n = *a, H_n = oracle_hubble(a_n, c);
    for (long long k = 0; k < M; ++k) {
        const double A = G * (acc[k] + B * pos[k]) / (a_n * a_n * a_n) - 2.0 * H_n * vel[k];
        vel[k] += A * (0.5 * dt);                                    /* Eq. 9  */
    }
    for (long long k = 0; k < M; ++k) pos[k] += vel[k] * dt;         /* Eq. 10 */
    const double a_1 = (c->H0 == 0.0) ? a_n : oracle_rk4_scale_factor(a_n, dt, c);
    const double H_1 = oracle_hubble(a_1, c);
    oracle_forces(pos, mass, soft, N, NULL, 0, acc, 0);
    for (long long k = 0; k < M; ++k) {
        /* v' = v + [G a^-3 g - 2 H v'] dt/2  solved for v' */
        const double g = G * (acc[k] + B * pos[k]) / (a_1 * a_1 * a_1);
        vel[k] = (vel[k] + g * (0.5 * dt)) / (1.0 + H_1 * dt);
    }
    *a = a_1;
}

/* The same step expressed as the coefficients the library's fused kick/drift kernel takes
 * (include/steps.h, steps_kdk_coeffs), derived here independently so the tests can
 * cross-check the host-side schedule:  v <- alpha v + beta (acc + B x),  x <- x + gamma v.
 * out = {alpha_open, beta_open, gamma, alpha_close, beta_close, a_next}. */
void oracle_kdk_coeffs(double a_n, double dt, double G, const oracle_cosmo *c, double *out)
{
    const double H_n = oracle_hubble(a_n, c);
    const double a_1 = (c->H0 == 0.0) ? a_n : oracle_rk4_scale_factor(a_n, dt, c);
    const double H_1 = oracle_hubble(a_1, c);
    out[0] = 1.0 - H_n * dt;
    out[1] = G / (a_n * a_n * a_n) * 0.5 * dt;
    out[2] = dt;
    out[3] = 1.0 / (1.0 + H_1 * dt);
    out[4] = G / (a_1 * a_1 * a_1) * 0.5 * dt / (1.0 + H_1 * dt);
    out[5] = a_1;
}

/* Literal-reading variant used only by the convergence pin that discriminates reading #8:
 * drag explicit in BOTH half kicks (first order in the drag). */
void oracle_kdk_step_explicit_drag(double *pos, double *vel, double *acc, const double *mass,
                                   const double *soft, long long N, double *a, double dt, double G,
                                   double B, const oracle_cosmo *c)
{
    const long long M = 3 * N;
    const double a_n = *a, H_n = oracle_hubble(a_n, c);
    for (long long k = 0; k < M; ++k)
        vel[k] += (G * (acc[k] + B * pos[k]) / (a_n * a_n * a_n) - 2.0 * H_n * vel[k]) * (0.5 * dt);
    for (long long k = 0; k < M; ++k) pos[k] += vel[k] * dt;
    const double a_1 = (c->H0 == 0.0) ? a_n : oracle_rk4_scale_factor(a_n, dt, c);
    const double H_1 = oracle_hubble(a_1, c);
    oracle_forces(pos, mass, soft, N, NULL, 0, acc, 0);
    for (long long k = 0; k < M; ++k)
        vel[k] += (G * (acc[k] + B * pos[k]) / (a_1 * a_1 * a_1) - 2.0 * H_1 * vel[k]) * (0.5 * dt);
    *a = a_1;
}

/* Diagnostics: P = sum m_i v_i  and  sum m_i |v_i|. */
void oracle_momentum(const double *vel, const double *mass, long long N, double *out4)
{
    double s[3] = {0, 0, 0}, c[3] = {0, 0, 0}, sa = 0, ca = 0;
    for (long long i = 0; i < N; ++i) {
        const double vx = vel[i], vy = vel[N + i], vz = vel[2 * N + i];
        neumaier_add(&s[0], &c[0], mass[i] * vx);
        neumaier_add(&s[1], &c[1], mass[i] * vy);
        neumaier_add(&s[2], &c[2], mass[i] * vz);
        neumaier_add(&sa, &ca, mass[i] * sqrt(vx * vx + vy * vy + vz * vz));
    }
    out4[0] = s[0] + c[0]; out4[1] = s[1] + c[1]; out4[2] = s[2] + c[2]; out4[3] = sa + ca;
}

/*
 * Adaptive time step, Eq. 12 (L113-116):
 *     dt = min[ dt_max, min_i sqrt( 2 eta_i eps / |A_i| ) ],   eta_i = 2.8 h_i  (L116, literal).
 * Readings (#11): one global step, the minimum over all particles (the integrator of Eq. 9-11 advances
 * every particle with the same dt); A_i is the acceleration that the kick applies, without the velocity-dependent
 * drag: A_i = coef (acc_i + B x_i) with coef = G a^-3 (Eq. 8, reading #6).  |A_i| = 0 puts no limit on dt.
 * Plain loop, fp64, in the order of the formula.
 */
double oracle_timestep(const double *pos, const double *acc, const double *soft, long long N, double coef, double B,
                       double eps, double dt_max)
{
    double dt = dt_max;
    for (long long i = 0; i < N; ++i) {
        const double Ax = coef * (acc[i] + B * pos[i]);
        const double Ay = coef * (acc[N + i] + B * pos[N + i]);
        const double Az = coef * (acc[2 * N + i] + B * pos[2 * N + i]);
        const double A = sqrt(Ax * Ax + Ay * Ay + Az * Az);
        if (A > 0.0) {
            const double eta = 2.8 * soft[i];
            const double dti = sqrt(2.0 * eta * eps / A);
            if (dti < dt) dt = dti;
        }
    }
    return dt;
}

/*
 * Net-force residual, the convergence monitor of glass generation (section 3.1 "the net gravitational
 * force acting on each particle is as small as possible"; L245 "integrating Eq. 8 with reversed gravity"):
 *     g_i = acc_i + B x_i        (the bracket of Eq. 8 L88 with reading #6: pair sum + background term, G = 1)
 *     out[0] = sum_i |g_i|^2     out[1] = max_i |g_i|
 * Neumaier-compensated sum, plain loop.  (Reversed gravity itself needs no function: it is G < 0 in the kick.)
 */
void oracle_force_residual(const double *pos, const double *acc, long long N, double B, double *out2)
{
    double s = 0.0, c = 0.0, mx = 0.0;
    for (long long i = 0; i < N; ++i) {
        const double gx = acc[i] + B * pos[i];
        const double gy = acc[N + i] + B * pos[N + i];
        const double gz = acc[2 * N + i] + B * pos[2 * N + i];
        const double g2 = gx * gx + gy * gy + gz * gz;
        neumaier_add(&s, &c, g2);
        const double g = sqrt(g2);
        if (g > mx) mx = g;
    }
    out2[0] = s + c;
    out2[1] = mx;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
