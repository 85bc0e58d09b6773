/*
 * gen_links.c -- seeded synthetic SU(3) lattice gauge fields (input generator).
 *
 * This module only MAKES INPUTS.  It holds none of the gauge-fixing method's arithmetic
 * (no Delta, no FFT, no link update) and is shared by the CPU oracle tests and the CUDA
 * path so that both see the same bytes.  It shares no code with oracle/ or with csrc/.
 *
 * Recipe (BASELINE.json `configs`):
 *   U_mu(x) = g0(x) exp(i sum_a w^a_mu(x) lambda_a / 2) g0(x+mu)^dagger
 *   w^a_mu(x) ~ N(0, sigma^2) i.i.d. per (x, mu, a);  lambda_a = Gell-Mann matrices;
 *   g0(x) Haar-random SU(3) per site (Ginibre matrix -> Gram-Schmidt, det fixed to +1).
 * The paper's own workloads (32^4 Wilson-action configurations, beta = 5.8..6.2,
 * PAPER.md:171) are not available; this generator stands in for them.
 *
 * Random numbers are counter based: every draw is a hash of (seed, stream, site, mu,
 * component, draw index), so the field does not depend on thread count or machine.
 *
 * Output layout (the library's interchange layout, include/lgf.h):
 *   out[(((s*4 + mu)*3 + row)*3 + col)*2 + {0:re,1:im}],  s = ix + Nx*(iy + Ny*(iz + Nz*it)).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stddef.h>

typedef double complex cd;

static inline uint64_t mix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* uniform in (0,1), 53 bits */
static inline double u01(uint64_t key, uint64_t counter)
{
    uint64_t r = mix64(key ^ mix64(counter));
    return ((double)(r >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* standard normal, Box-Muller on two counter-indexed uniforms */
static inline double normal(uint64_t key, uint64_t counter)
{
    double u1 = u01(key, 2 * counter), u2 = u01(key, 2 * counter + 1);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

static void matmul3(const cd a[9], const cd b[9], cd c[9])
{
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            cd s = 0;
            for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
            c[3 * i + j] = s;
        }
}

/* make m special unitary: normalise row 0, orthonormalise row 1, row 2 = conj(row0 x row1) */
static void su3_cleanup(cd m[9])
{
    double n0 = 0;
    for (int j = 0; j < 3; j++) n0 += creal(m[j] * conj(m[j]));
    n0 = 1.0 / sqrt(n0);
    for (int j = 0; j < 3; j++) m[j] *= n0;
    cd p = 0;
    for (int j = 0; j < 3; j++) p += conj(m[j]) * m[3 + j];
    for (int j = 0; j < 3; j++) m[3 + j] -= p * m[j];
    double n1 = 0;
    for (int j = 0; j < 3; j++) n1 += creal(m[3 + j] * conj(m[3 + j]));
    n1 = 1.0 / sqrt(n1);
    for (int j = 0; j < 3; j++) m[3 + j] *= n1;
    m[6] = conj(m[1] * m[5] - m[2] * m[4]);
    m[7] = conj(m[2] * m[3] - m[0] * m[5]);
    m[8] = conj(m[0] * m[4] - m[1] * m[3]);
}

/* H = sum_a w[a] lambda_a / 2 with the standard Gell-Mann matrices (Tr la lb = 2 dab) */
static void gellmann_sum(const double w[8], cd h[9])
{
    const double r3 = 0.57735026918962576450914878050196; /* 1/sqrt(3) */
    h[0] = 0.5 * (w[2] + r3 * w[7]);
    h[4] = 0.5 * (-w[2] + r3 * w[7]);
    h[8] = 0.5 * (-2.0 * r3 * w[7]);
    h[1] = 0.5 * (w[0] - I * w[1]);
    h[3] = 0.5 * (w[0] + I * w[1]);
    h[2] = 0.5 * (w[3] - I * w[4]);
    h[6] = 0.5 * (w[3] + I * w[4]);
    h[5] = 0.5 * (w[5] - I * w[6]);
    h[7] = 0.5 * (w[5] + I * w[6]);
}

/* e = exp(i h), h Hermitian traceless: scaling and squaring + Taylor, then clean-up */
static void exp_i_herm(const cd h[9], cd e[9])
{
    double nrm = 0;
    for (int k = 0; k < 9; k++) nrm += cabs(h[k]);
    int sq = 0;
    while (nrm > 0.125 && sq < 60) { nrm *= 0.5; sq++; }
    double sc = ldexp(1.0, -sq);
    cd a[9], term[9], tmp[9];
    for (int k = 0; k < 9; k++) a[k] = I * h[k] * sc;
    for (int k = 0; k < 9; k++) { e[k] = (k % 4 == 0) ? 1.0 : 0.0; term[k] = e[k]; }
    for (int n = 1; n <= 18; n++) {
        matmul3(term, a, tmp);
        for (int k = 0; k < 9; k++) { term[k] = tmp[k] / (double)n; e[k] += term[k]; }
    }
    for (int s = 0; s < sq; s++) {
        matmul3(e, e, tmp);
        for (int k = 0; k < 9; k++) e[k] = tmp[k];
    }
    su3_cleanup(e);
}

static void haar_su3(uint64_t key, uint64_t site, cd g[9])
{
    for (int k = 0; k < 9; k++) {
        double re = normal(key, site * 18 + 2 * k), im = normal(key, site * 18 + 2 * k + 1);
        g[k] = re + I * im;
    }
    su3_cleanup(g);
}

/*
 * Haar-random g0 per site.  out_g[(s*9 + 3*row + col)*2 + {re,im}].
 */
void gen_haar_field(const int N[4], uint64_t seed, double *out_g)
{
    const int64_t V = (int64_t)N[0] * N[1] * N[2] * N[3];
    const uint64_t kg = mix64(seed ^ 0x6730ULL);
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < V; s++) {
        cd g[9];
        haar_su3(kg, (uint64_t)s, g);
        for (int k = 0; k < 9; k++) {
            out_g[(s * 9 + k) * 2] = creal(g[k]);
            out_g[(s * 9 + k) * 2 + 1] = cimag(g[k]);
        }
    }
}

/*
 * The BASELINE.json recipe.  sigma = 0 gives a pure-gauge field (a Haar-random gauge
 * transform of the unit field).  haar = 0 skips the gauge transform (g0 = 1).
 */
void gen_links(const int N[4], double sigma, uint64_t seed, int haar, double *out)
{
    const int64_t V = (int64_t)N[0] * N[1] * N[2] * N[3];
    const uint64_t kw = mix64(seed ^ 0x7711ULL), kg = mix64(seed ^ 0x6730ULL);
    const int64_t stride[4] = {1, N[0], (int64_t)N[0] * N[1], (int64_t)N[0] * N[1] * N[2]};
#pragma omp parallel for schedule(static)
    for (int64_t s = 0; s < V; s++) {
        int c[4];
        int64_t r = s;
        for (int d = 0; d < 4; d++) { c[d] = (int)(r % N[d]); r /= N[d]; }
        cd g0[9];
        if (haar) haar_su3(kg, (uint64_t)s, g0);
        for (int mu = 0; mu < 4; mu++) {
            double w[8];
            for (int a = 0; a < 8; a++)
                w[a] = sigma * normal(kw, ((uint64_t)s * 4 + mu) * 8 + a);
            cd h[9], v[9], u[9];
            gellmann_sum(w, h);
            exp_i_herm(h, v);
            if (haar) {
                int64_t sp = s + ((c[mu] + 1 == N[mu]) ? -(int64_t)(N[mu] - 1) : 1) * stride[mu];
                cd g1[9], g1d[9], t[9];
                haar_su3(kg, (uint64_t)sp, g1);
                for (int i = 0; i < 3; i++)
                    for (int j = 0; j < 3; j++) g1d[3 * i + j] = conj(g1[3 * j + i]);
                matmul3(g0, v, t);
                matmul3(t, g1d, u);
            } else {
                for (int k = 0; k < 9; k++) u[k] = v[k];
            }
            double *o = out + ((s * 4 + mu) * 9) * 2;
            for (int k = 0; k < 9; k++) { o[2 * k] = creal(u[k]); o[2 * k + 1] = cimag(u[k]); }
        }
    }
}
