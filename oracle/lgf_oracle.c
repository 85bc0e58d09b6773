/*
 * lgf_oracle.c -- CPU ORACLE for the Fourier-accelerated steepest-descent SU(3) Landau
 * gauge fixing iteration of arXiv 1210.8018 (Algorithm 1).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It is plain, slow,
 * single-threaded FP64 C that follows the paper step by step, in the paper's order and
 * notation, so that it can be checked against the paper by eye.  It shares no code with
 * the CUDA path (paper_1210_8018_b200/csrc) nor with the input generator (gen/).
 *
 * Layouts (all AoS, `double complex`):
 *   site index   s = ix + Nx*(iy + Ny*(iz + Nz*it)),  N[0..3] = Nx,Ny,Nz,Nt, mu=0..3 <-> x,y,z,t
 *   links        U[(s*4 + mu)*9 + 3*row + col]
 *   site fields  Delta, w, g:  X[s*9 + 3*row + col]
 *   scalar field f[s]
 *
 * Steps:
 *   O0 orc_momentum_tables / orc_mask     p^2 = eigenvalues of -d^2, eq. 1.2
 *   O1 orc_measure                        eq. 1.5, eq. 1.1 at g=1, eq. 1.4
 *   O3 orc_fft4d(sign=-1)                 Alg. 1 "apply FFT forward"
 *   O4 multiply by orc_mask               Alg. 1 "apply p_max^2/p^2"
 *   O5 orc_fft4d(sign=+1), times 1/V      Alg. 1 "apply FFT backward", "normalize"
 *   O6 orc_build_g                        "expand the exponential to first order in alpha, followed by
 *                                          a reunitarization"; Alg. 1 lines 9-11
 *   O7 orc_update_links                   U_mu(x) -> g(x) U_mu(x) g^dagger(x+mu)
 *   O2/O8 orc_fix                         while theta > eps
 *
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md (R1-R21).
 * Pins: tests/test_oracle_*.py (closed forms, brute-force DFT, numpy.fft, invariants).
 * Parity unpinned: the numerical VALUES of F, theta and iteration counts on a given input
 * (the paper prints none); they are pinned only through the invariants above.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cd;
#define NC 3
static const double TWO_PI = 6.283185307179586476925286766559;

static int64_t volume(const int N[4]) { return (int64_t)N[0] * N[1] * N[2] * N[3]; }

static void coords(const int N[4], int64_t s, int c[4])
{
    for (int d = 0; d < 4; d++) { c[d] = (int)(s % N[d]); s /= N[d]; }
}

static int64_t site(const int N[4], const int c[4])
{
    return c[0] + (int64_t)N[0] * (c[1] + (int64_t)N[1] * (c[2] + (int64_t)N[2] * c[3]));
}

/* index of x + dir*mu_hat with periodic wrap, dir = +1 or -1 */
static int64_t neighbour(const int N[4], int64_t s, int mu, int dir)
{
    int c[4];
    coords(N, s, c);
    c[mu] = (c[mu] + dir + N[mu]) % N[mu];
    return site(N, c);
}

/* ------------------------------------------------------------------ O0: tables */

/* s_mu[k] = 4 sin^2(pi k / N_mu): eigenvalues of minus the lattice second difference along
 * mu ("p^2 are the eigenvalues of (-d^2)", lattice spacing a = 1; reading R5).
 * tab holds the four tables back to back: N[0] + N[1] + N[2] + N[3] doubles.
 * *pmax2 = max_k p^2(k) = sum_mu max_k s_mu[k] (reading R6). */
void orc_momentum_tables(const int N[4], double *tab, double *pmax2)
{
    double pm = 0;
    int off = 0;
    for (int mu = 0; mu < 4; mu++) {
        double m = 0;
        for (int k = 0; k < N[mu]; k++) {
            double sn = sin(0.5 * TWO_PI * (double)k / (double)N[mu]);
            tab[off + k] = 4.0 * sn * sn;
            if (tab[off + k] > m) m = tab[off + k];
        }
        pm += m;
        off += N[mu];
    }
    *pmax2 = pm;
}

/* M(k) = p_max^2 / p^2(k), with the zero mode set to 0 (eq. 1.2; reading R7). */
void orc_mask(const int N[4], double *M)
{
    int ntab = N[0] + N[1] + N[2] + N[3];
    double *tab = malloc(sizeof(double) * ntab), pmax2;
    orc_momentum_tables(N, tab, &pmax2);
    const double *s0 = tab, *s1 = s0 + N[0], *s2 = s1 + N[1], *s3 = s2 + N[2];
    int64_t V = volume(N);
    for (int64_t k = 0; k < V; k++) {
        int c[4];
        coords(N, k, c);
        double p2 = s0[c[0]] + s1[c[1]] + s2[c[2]] + s3[c[3]];
        M[k] = (k == 0) ? 0.0 : pmax2 / p2;
    }
    free(tab);
}

/* ------------------------------------------------------------------ O1: measure */

/* Delta(x) = sum_nu [ U_nu(x - nu) - U_nu(x) - h.c. - trace ]           (eq. 1.5)
 *   A = sum_nu [U_nu(x-nu) - U_nu(x)];  D = A - A^dagger;  Delta = D - (Tr D / N_c) 1  (reading R3)
 * F = 1/(4 N_c V) sum_x sum_mu Re Tr U_mu(x)                            (eq. 1.1 at g = 1)
 * theta = 1/(N_c V) sum_x Tr[Delta Delta^dagger]                        (eq. 1.4)
 * Delta may be NULL. */
void orc_measure(const int N[4], const cd *U, cd *Delta, double *F, double *theta)
{
    int64_t V = volume(N);
    long double sumF = 0, sumT = 0;
    for (int64_t x = 0; x < V; x++) {
        cd A[9], D[9];
        for (int k = 0; k < 9; k++) A[k] = 0;
        for (int nu = 0; nu < 4; nu++) {
            int64_t xm = neighbour(N, x, nu, -1);
            const cd *Ub = U + (xm * 4 + nu) * 9, *Uf = U + (x * 4 + nu) * 9;
            for (int k = 0; k < 9; k++) A[k] += Ub[k] - Uf[k];
            sumF += creal(Uf[0] + Uf[4] + Uf[8]);
        }
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) D[3 * i + j] = A[3 * i + j] - conj(A[3 * j + i]);
        cd tr = (D[0] + D[4] + D[8]) / (double)NC;
        D[0] -= tr; D[4] -= tr; D[8] -= tr;
        for (int k = 0; k < 9; k++) sumT += creal(D[k] * conj(D[k]));
        if (Delta) for (int k = 0; k < 9; k++) Delta[x * 9 + k] = D[k];
    }
    *F = (double)(sumF / (4.0L * NC * (long double)V));
    *theta = (double)(sumT / ((long double)NC * (long double)V));
}

/* ------------------------------------------------------------------ O3/O5: FFT */

/* exp(sign * 2 pi i k / n), evaluated directly for each k (no recurrence) */
static cd root_of_unity(int n, int k, int sign)
{
    k %= n;
    double a = TWO_PI * (double)k / (double)n;
    return cos(a) + I * (sign * sin(a));
}

/* Textbook iterative radix-2 decimation-in-time FFT, n a power of two, in place:
 * bit-reversal permutation, then log2(n) butterfly stages. */
static void fft_radix2(int n, cd *x, int sign)
{
    cd *W = malloc(sizeof(cd) * n);              /* W[k] = exp(sign 2 pi i k / n), each k directly */
    for (int k = 0; k < n; k++) W[k] = root_of_unity(n, k, sign);
    for (int i = 1, j = 0; i < n; i++) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cd t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        for (int i = 0; i < n; i += len)
            for (int k = 0; k < len / 2; k++) {
                cd w = W[k * (n / len)];         /* = exp(sign 2 pi i k / len) */
                cd u = x[i + k], v = w * x[i + k + len / 2];
                x[i + k] = u + v;
                x[i + k + len / 2] = u - v;
            }
    }
    free(W);
}

/* Textbook recursive Cooley-Tukey on the smallest prime factor p of n (n = p*m):
 * X[k + m*q] = sum_r W_n^{r(k + m q)} Y_r[k],  Y_r = DFT_m of x[p*j + r].
 * For prime n this is the direct O(n^2) DFT.  out must not alias in. */
static void fft_mixed(int n, const cd *in, int stride, cd *out, int sign)
{
    if (n == 1) { out[0] = in[0]; return; }
    int p = 2;
    while (n % p) p++;
    int m = n / p;
    cd *Y = malloc(sizeof(cd) * n);
    for (int r = 0; r < p; r++) fft_mixed(m, in + (int64_t)r * stride, stride * p, Y + r * m, sign);
    for (int k = 0; k < m; k++)
        for (int q = 0; q < p; q++) {
            cd s = 0;
            for (int r = 0; r < p; r++) s += root_of_unity(n, (r * (k + m * q)) % n, sign) * Y[r * m + k];
            out[k + m * q] = s;
        }
    free(Y);
}

/* 1D unnormalised DFT: X[k] = sum_j x[j] exp(sign 2 pi i j k / n); sign = -1 forward, +1 backward */
void orc_fft1d(int n, cd *x, int sign)
{
    if ((n & (n - 1)) == 0) { fft_radix2(n, x, sign); return; }
    cd *tmp = malloc(sizeof(cd) * n);
    fft_mixed(n, x, 1, tmp, sign);
    memcpy(x, tmp, sizeof(cd) * n);
    free(tmp);
}

/* 4D unnormalised DFT of a scalar field: four passes of 1D transforms, one per axis
 * (reading R8: forward e^{-i}, backward e^{+i}, 1/V applied by the caller). */
void orc_fft4d(const int N[4], cd *f, int sign)
{
    int64_t V = volume(N);
    int64_t stride = 1;
    for (int mu = 0; mu < 4; mu++) {
        int n = N[mu];
        cd *line = malloc(sizeof(cd) * n);
        for (int64_t s = 0; s < V; s++) {
            int c[4];
            coords(N, s, c);
            if (c[mu] != 0) continue;           /* s is the start of a line along mu */
            for (int j = 0; j < n; j++) line[j] = f[s + j * stride];
            orc_fft1d(n, line, sign);
            for (int j = 0; j < n; j++) f[s + j * stride] = line[j];
        }
        free(line);
        stride *= n;
    }
}

/* Alg. 1 lines 3-8: for every element (i,j) of the Delta(x) matrix:
 * FFT forward, apply p_max^2/p^2, FFT backward, normalise by 1/V.  All 9 elements (reading R9). */
void orc_fourier_accelerate(const int N[4], const cd *Delta, cd *w)
{
    int64_t V = volume(N);
    double *M = malloc(sizeof(double) * V);
    cd *f = malloc(sizeof(cd) * V);
    orc_mask(N, M);
    for (int e = 0; e < 9; e++) {
        for (int64_t x = 0; x < V; x++) f[x] = Delta[x * 9 + e];
        orc_fft4d(N, f, -1);
        for (int64_t k = 0; k < V; k++) f[k] *= M[k];
        orc_fft4d(N, f, +1);
        for (int64_t x = 0; x < V; x++) w[x * 9 + e] = f[x] / (double)V;
    }
    free(f);
    free(M);
}

/* ------------------------------------------------------------------ O6: g(x) */

/* g(x) = reunit( 1 + (alpha/2) w(x) )  (first order of eq. 1.2; R10, R11).
 * Reunitarisation = Gram-Schmidt on rows 0, 1; row 2 = conj(row0 x row1)  (readings R12, R13):
 *   u = m_0 / |m_0|;  v' = m_1 - <u, m_1> u with <u, m_1> = sum_j conj(u_j) m_1j;  v = v'/|v'|;
 *   t_i = conj( eps_ijk u_j v_k ). */
void orc_build_g(int64_t V, const cd *w, double alpha, cd *g)
{
    for (int64_t x = 0; x < V; x++) {
        cd m[9];
        for (int k = 0; k < 9; k++) m[k] = ((k % 4 == 0) ? 1.0 : 0.0) + (alpha / 2.0) * w[x * 9 + k];
        cd u[3], v[3], t[3];
        double nu = 0;
        for (int j = 0; j < 3; j++) nu += creal(m[j] * conj(m[j]));
        nu = sqrt(nu);
        for (int j = 0; j < 3; j++) u[j] = m[j] / nu;
        cd ip = 0;
        for (int j = 0; j < 3; j++) ip += conj(u[j]) * m[3 + j];
        for (int j = 0; j < 3; j++) v[j] = m[3 + j] - ip * u[j];
        double nv = 0;
        for (int j = 0; j < 3; j++) nv += creal(v[j] * conj(v[j]));
        nv = sqrt(nv);
        for (int j = 0; j < 3; j++) v[j] /= nv;
        t[0] = conj(u[1] * v[2] - u[2] * v[1]);
        t[1] = conj(u[2] * v[0] - u[0] * v[2]);
        t[2] = conj(u[0] * v[1] - u[1] * v[0]);
        for (int j = 0; j < 3; j++) { g[x * 9 + j] = u[j]; g[x * 9 + 3 + j] = v[j]; g[x * 9 + 6 + j] = t[j]; }
    }
}

/* Variant named by the paper: eq. 1.2 as written, g(x) = exp[(alpha/2) w(x)]
 * (PAPER.md:49), instead of its first-order expansion followed by a reunitarisation.
 * Textbook scaling and squaring: B = A / 2^s with |B|_F <= 1/4, exp(B) by its Taylor series
 * summed until the terms vanish in FP64, then s squarings.  A = (alpha/2) w is anti-Hermitian and
 * traceless, so exp(A) is in SU(3) up to rounding; no projection is applied. */
void orc_build_g_exp(int64_t V, const cd *w, double alpha, cd *g)
{
    for (int64_t x = 0; x < V; x++) {
        cd A[9], E[9], term[9], tmp[9];
        double nrm = 0;
        for (int k = 0; k < 9; k++) { A[k] = (alpha / 2.0) * w[x * 9 + k]; nrm += creal(A[k] * conj(A[k])); }
        nrm = sqrt(nrm);
        int s = 0;
        while (nrm > 0.25) { nrm *= 0.5; s++; }
        for (int k = 0; k < 9; k++) { A[k] = ldexp(creal(A[k]), -s) + I * ldexp(cimag(A[k]), -s); }
        for (int k = 0; k < 9; k++) { E[k] = (k % 4 == 0) ? 1.0 : 0.0; term[k] = E[k]; }
        for (int n = 1; n <= 40; n++) {
            /* term <- term A / n */
            double tn = 0;
            for (int i = 0; i < 3; i++)
                for (int j = 0; j < 3; j++) {
                    cd a = 0;
                    for (int k = 0; k < 3; k++) a += term[3 * i + k] * A[3 * k + j];
                    tmp[3 * i + j] = a / (double)n;
                    tn += creal(tmp[3 * i + j] * conj(tmp[3 * i + j]));
                }
            for (int k = 0; k < 9; k++) { term[k] = tmp[k]; E[k] += term[k]; }
            if (tn < 1e-40) break;
        }
        for (int q = 0; q < s; q++) {
            for (int i = 0; i < 3; i++)
                for (int j = 0; j < 3; j++) {
                    cd a = 0;
                    for (int k = 0; k < 3; k++) a += E[3 * i + k] * E[3 * k + j];
                    tmp[3 * i + j] = a;
                }
            for (int k = 0; k < 9; k++) E[k] = tmp[k];
        }
        for (int k = 0; k < 9; k++) g[x * 9 + k] = E[k];
    }
}

/* ------------------------------------------------------------------ O7: link update */

static void mul3(const cd *a, const cd *b, cd *c) /* c = a b */
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cd s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}

static void mul3_dag(const cd *a, const cd *b, cd *c) /* c = a b^dagger */
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cd s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * conj(b[3 * j + k]);
            c[3 * i + j] = s;
        }
}

/* U_mu(x) -> g(x) U_mu(x) g^dagger(x + mu) for all x, mu (Alg. 1 lines 12-16).
 * All g are given (computed from the old Delta), so the order of sites is immaterial (R14). */
void orc_update_links(const int N[4], cd *U, const cd *g)
{
    int64_t V = volume(N);
    for (int64_t x = 0; x < V; x++)
        for (int mu = 0; mu < 4; mu++) {
            int64_t xp = neighbour(N, x, mu, +1);
            cd t[9], r[9];
            mul3(g + x * 9, U + (x * 4 + mu) * 9, t);
            mul3_dag(t, g + xp * 9, r);
            memcpy(U + (x * 4 + mu) * 9, r, sizeof r);
        }
}

/* ------------------------------------------------------------------ Algorithm 1 */

/* One pass of the loop body (Alg. 1 lines 3-16) given Delta of the current links. */
static int g_mode = 0; /* 0: first order + reunitarisation (the paper's choice); 1: exact exponential */

/* Select how g(x) is formed in orc_iterate / orc_fix (single-threaded test infrastructure: a plain global). */
void orc_set_exponential(int on) { g_mode = on ? 1 : 0; }

static void loop_body(const int N[4], cd *U, const cd *Delta, double alpha, cd *w, cd *g)
{
    orc_fourier_accelerate(N, Delta, w);
    if (g_mode) orc_build_g_exp(volume(N), w, alpha, g);
    else orc_build_g(volume(N), w, alpha, g);
    orc_update_links(N, U, g);
}

/* Exactly n iterations, ignoring theta.  hist (may be NULL) receives (F, theta) after the
 * initial measure and after every iteration: 2*(n+1) doubles. */
void orc_iterate(const int N[4], cd *U, double alpha, int64_t n, double *hist)
{
    int64_t V = volume(N);
    cd *Delta = malloc(sizeof(cd) * 9 * V), *w = malloc(sizeof(cd) * 9 * V), *g = malloc(sizeof(cd) * 9 * V);
    double F, theta;
    orc_measure(N, U, Delta, &F, &theta);
    if (hist) { hist[0] = F; hist[1] = theta; }
    for (int64_t it = 1; it <= n; it++) {
        loop_body(N, U, Delta, alpha, w, g);
        orc_measure(N, U, Delta, &F, &theta);
        if (hist) { hist[2 * it] = F; hist[2 * it + 1] = theta; }
    }
    free(Delta); free(w); free(g);
}

/* Algorithm 1: measure; while theta > eps (reading R2: stop when
 * theta <= eps): loop body; measure.  Returns the number of executions of the
 * loop body (reading R16), or -1 if max_iter was reached first.  F, theta are those of the
 * final links.  hist (may be NULL) receives (F, theta) of iteration 0, 1, ... while there is
 * room (hist_cap pairs). */
int64_t orc_fix(const int N[4], cd *U, double alpha, double eps, int64_t max_iter,
                double *F, double *theta, double *hist, int64_t hist_cap)
{
    int64_t V = volume(N);
    cd *Delta = malloc(sizeof(cd) * 9 * V), *w = malloc(sizeof(cd) * 9 * V), *g = malloc(sizeof(cd) * 9 * V);
    int64_t it = 0;
    orc_measure(N, U, Delta, F, theta);
    if (hist && hist_cap > 0) { hist[0] = *F; hist[1] = *theta; }
    while (*theta > eps) {
        if (it >= max_iter) { it = -1; break; }
        loop_body(N, U, Delta, alpha, w, g);
        orc_measure(N, U, Delta, F, theta);
        it++;
        if (hist && it < hist_cap) { hist[2 * it] = *F; hist[2 * it + 1] = *theta; }
    }
    free(Delta); free(w); free(g);
    return it;
}

/* ------------------------------------------------------------------ invariant used by the pins */

/* Average plaquette 1/(6 N_c V) sum_x sum_{mu<nu} Re Tr[U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)].
 * Gauge invariant; not part of Algorithm 1, used only to pin orc_update_links (pin P11). */
double orc_plaquette(const int N[4], const cd *U)
{
    int64_t V = volume(N);
    long double sum = 0;
    for (int64_t x = 0; x < V; x++)
        for (int mu = 0; mu < 4; mu++)
            for (int nu = mu + 1; nu < 4; nu++) {
                int64_t xmu = neighbour(N, x, mu, +1), xnu = neighbour(N, x, nu, +1);
                cd a[9], b[9], c[9];
                mul3(U + (x * 4 + mu) * 9, U + (xmu * 4 + nu) * 9, a);
                mul3_dag(a, U + (xnu * 4 + mu) * 9, b);
                mul3_dag(b, U + (x * 4 + nu) * 9, c);
                sum += creal(c[0] + c[4] + c[8]);
            }
    return (double)(sum / (6.0L * NC * (long double)V));
}
