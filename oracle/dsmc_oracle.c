/*
 * dsmc_oracle.c -- plain fp64 CPU ORACLE for the hot path of arXiv 1211.6234
 * (Stamps & Ambrose): lattice-summed dipole tensor W, dipole field h = W (*) s,
 * energy, Philox-driven checkerboard Metropolis half-sweep with the paper's
 * frozen-field approximation, observables.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check in
 * __graft_entry__.py and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.  It shares no code, header, table or constant
 * generator with paper_1211_6234_b200/csrc (the CUDA path) and neither includes
 * the other.  Everything is written the slow, obvious way, in the paper's order
 * and notation, so that it can be checked against PAPER.md by eye.  The only
 * concession to run time is "#pragma omp parallel for" on outermost loops whose
 * iterations are independent (no blocking, no fusion, no reordering of sums).
 *
 * Citations are PAPER.md:<line> (section / equation) and DESIGN.md "Readings"
 * (R-numbers) for points where the paper is silent, garbled or ambiguous.
 *
 * Conventions:
 *   lattice site n = (x, y), x, y in [0, L), linear index n = y*L + x  (PAPER.md:325,
 *   App. A "j = S_y L + S_x").  N = L*L.  k_B = 1, energies in units of J.
 *   spins   s[r][c][y][x]   r in [0,R), c in {x,y,z}      (fp64, unit vectors)
 *   tensor  W[c][rho_y][rho_x], c in {xx, xy, yy, zz}, rho = (m - n) mod L
 *   field   h[r][c][y][x]   in lattice units (no factor g)
 *   E = -J sum_bonds s.s - sum_n (K2 s_z^2 + K4 s_z^4) + (g/2) sum_n s_n . h_n   (R7)
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   build_tensor_*  : Laplace invariant, D4 symmetries, closed-form lattice sums
 *                     4 zeta(3/2) beta(3/2), two independent routes (image+tail vs
 *                     Ewald), Ewald independent of the splitting parameter.
 *   dipole_field / energy : brute-force eq. 1 with explicit images on L <= 4;
 *                     uniform and alternating states against closed forms.
 *   philox4x32_10   : published known-answer vectors (Salmon et al., SC'11).
 *   delta_e / halfsweep : single-spin dE == full-energy difference; eq. 8 identity;
 *                     g = 0 limit; T -> infinity and T -> 0 limits.
 *   halfsweep_sequential : g = 0 equals the frozen sweep; g != 0: the eq. 8 terms of the
 *                     sites updated before, term by term.
 *   *_given_field   : identical to the plain calls when handed the plain field.
 *   observables     : cone-angle special cases of PAPER.md:241, :255.
 *   eq. 10's "0.14 %" is NOT reproduced: parity unpinned for that
 *   number (context only, nothing on the hot path depends on it).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* O1. The interaction table W (eq. 1-2).                     */
/* ------------------------------------------------------------------------- */

/* Bracket of eq. 1 for one pair at in-plane separation r=(x,y,0):
 *   T^{ab}(r) = (delta_ab - 3 rhat_a rhat_b) / r^3 .
 * With z = 0 the xz and yz components vanish; out = {xx, xy, yy, zz}.          */
static void pair_tensor(double x, double y, double out[4])
{
    double r2 = x * x + y * y;
    double r = sqrt(r2);
    double r3 = r2 * r;
    out[0] = (1.0 - 3.0 * (x / r) * (x / r)) / r3;
    out[1] = (-3.0 * (x / r) * (y / r)) / r3;
    out[2] = (1.0 - 3.0 * (y / r) * (y / r)) / r3;
    out[3] = 1.0 / r3;
}

/* reduce a displacement in [0, L) to the symmetric cell (-L/2, L/2]  (R3) */
static int reduce_sym(int rho, int L)
{
    return (rho <= L / 2) ? rho : rho - L;
}

/* Image route (BASELINE config 1: "image cutoff |a|,|b| <= 64"):
 *   W^{ab}(rho) = sum_{G=(aL,bL), |a|,|b|<=A} T^{ab}(rho + G),
 * the G = 0 term omitted when rho = 0 (the self-image term of eq. 2, PAPER.md:35,
 * read with coefficient 1/2 like every other pair: R2).
 * tail != 0 adds the remainder of the square cutoff treated as a continuum of
 * unit density: integral of r^-3 outside the square of half-side (A+1/2)L,
 *   t = 4 sqrt(2) / ((A + 1/2) L^3),
 * which goes to zz as +t and, by symmetry of the square and tracelessness of T,
 * to xx and yy as -t/2 each; xy gets 0.  (R6)                                   */
int oracle_build_tensor_image(int L, int A, int tail, double *W)
{
    if (L < 1 || A < 0 || !W) return -1;
    size_t N = (size_t)L * L;
#pragma omp parallel for schedule(dynamic, 1)
    for (int ry = 0; ry < L; ++ry) {
        for (int rx = 0; rx < L; ++rx) {
            int dx = reduce_sym(rx, L), dy = reduce_sym(ry, L);
            double acc[4] = {0, 0, 0, 0};
            for (int b = -A; b <= A; ++b) {
                for (int a = -A; a <= A; ++a) {
                    double x = (double)dx + (double)a * L;
                    double y = (double)dy + (double)b * L;
                    if (x == 0.0 && y == 0.0) continue;
                    double t[4];
                    pair_tensor(x, y, t);
                    for (int c = 0; c < 4; ++c) acc[c] += t[c];
                }
            }
            if (tail) {
                double t = 4.0 * sqrt(2.0) / (((double)A + 0.5) * (double)L * L * L);
                acc[0] -= 0.5 * t;
                acc[2] -= 0.5 * t;
                acc[3] += t;
            }
            for (int c = 0; c < 4; ++c) W[c * N + (size_t)ry * L + rx] = acc[c];
        }
    }
    return 0;
}

/* Ewald route (eq. 3-5; Harris' 2-D form), at z = z_nm = 0.
 * The extraction of eq. 3-5 is garbled (R4); restated with alpha = 1/(2 eta):
 *   1/r = erfc(alpha r)/r + erf(alpha r)/r,   T^{ab} = -d_a d_b (1/r).
 * Short-range part (eq. 3, f_S), -d_a d_b applied to erfc(alpha r)/r:
 *   delta_ab B(r) - r_a r_b C(r),
 *   B = erfc(alpha r)/r^3 + (2 alpha/sqrt(pi)) exp(-alpha^2 r^2)/r^2,
 *   C = 3 erfc(alpha r)/r^5 + (2 alpha/sqrt(pi)) (2 alpha^2 + 3/r^2) exp(-alpha^2 r^2)/r^2,
 *   summed over G (zz: only B, because z = 0).
 * Long-range part (eq. 4-5, f_L) with k = 2 pi (n_x, n_y)/L, cell area L^2:
 *   htilde(k, z=0) = (2 pi / k) erfc(k eta);
 *   in-plane a,b:  L^-2 sum_{k != 0} (2 pi k_a k_b / k) erfc(k eta) cos(k.rho)
 *   zz (needs d_z^2 of eq. 5's bracket at z = 0, which is why the paper keeps z,
 *   PAPER.md:44):  L^-2 sum_k [ (2 sqrt(pi)/eta) exp(-k^2 eta^2) - 2 pi k erfc(k eta) ] cos(k.rho),
 *   the k = 0 term (2 sqrt(pi)/eta)/L^2 is kept.
 * Self site rho = 0: drop G = 0 from the short-range sum and subtract the G = 0
 * piece of the long-range function, -d_a d_b [erf(alpha r)/r] at r = 0
 *   = (4 alpha^3 / (3 sqrt(pi))) delta_ab .
 * alphaL = alpha * L (any value in about [2, 4]: the result does not depend on it, R5);
 * nreal = image cutoff of the short-range sum, nk = cutoff of the k sum.          */
int oracle_build_tensor_ewald(int L, double alphaL, int nreal, int nk, double *W)
{
    if (L < 1 || !(alphaL > 0) || nreal < 0 || nk < 0 || !W) return -1;
    size_t N = (size_t)L * L;
    const double alpha = alphaL / (double)L;
    const double eta = 1.0 / (2.0 * alpha);
    const double two_a_sqrtpi = 2.0 * alpha / sqrt(ORACLE_PI);
    const double area = (double)L * (double)L;
#pragma omp parallel for schedule(dynamic, 1)
    for (int ry = 0; ry < L; ++ry) {
        for (int rx = 0; rx < L; ++rx) {
            int dx = reduce_sym(rx, L), dy = reduce_sym(ry, L);
            double acc[4] = {0, 0, 0, 0};
            /* f_S: short-range real-space sum */
            for (int b = -nreal; b <= nreal; ++b) {
                for (int a = -nreal; a <= nreal; ++a) {
                    double x = (double)dx + (double)a * L;
                    double y = (double)dy + (double)b * L;
                    if (x == 0.0 && y == 0.0) continue;
                    double r2 = x * x + y * y, r = sqrt(r2);
                    double ec = erfc(alpha * r), ex = exp(-alpha * alpha * r2);
                    double B = ec / (r2 * r) + two_a_sqrtpi * ex / r2;
                    double C = 3.0 * ec / (r2 * r2 * r) +
                               two_a_sqrtpi * (2.0 * alpha * alpha + 3.0 / r2) * ex / r2;
                    acc[0] += B - x * x * C;
                    acc[1] += -x * y * C;
                    acc[2] += B - y * y * C;
                    acc[3] += B;
                }
            }
            /* f_L: long-range Fourier sum */
            for (int ny = -nk; ny <= nk; ++ny) {
                for (int nx = -nk; nx <= nk; ++nx) {
                    double kx = 2.0 * ORACLE_PI * nx / (double)L;
                    double ky = 2.0 * ORACLE_PI * ny / (double)L;
                    double k = sqrt(kx * kx + ky * ky);
                    if (nx == 0 && ny == 0) {
                        acc[3] += (2.0 * sqrt(ORACLE_PI) / eta) / area;
                        continue;
                    }
                    double c = cos(kx * dx + ky * dy);
                    double ec = erfc(k * eta);
                    double f = 2.0 * ORACLE_PI * ec / k / area;
                    acc[0] += f * kx * kx * c;
                    acc[1] += f * kx * ky * c;
                    acc[2] += f * ky * ky * c;
                    acc[3] += ((2.0 * sqrt(ORACLE_PI) / eta) * exp(-k * k * eta * eta) -
                               2.0 * ORACLE_PI * k * ec) * c / area;
                }
            }
            if (rx == 0 && ry == 0) {
                double self = 4.0 * alpha * alpha * alpha / (3.0 * sqrt(ORACLE_PI));
                acc[0] -= self;
                acc[2] -= self;
                acc[3] -= self;
            }
            for (int c = 0; c < 4; ++c) W[c * N + (size_t)ry * L + rx] = acc[c];
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O2. Dipole field: plain definition (App. A :331-350).      */
/*   h_n^x = sum_m [ W^xx(rho_nm) s_m^x + W^xy(rho_nm) s_m^y ]                 */
/*   h_n^y = sum_m [ W^xy s_m^x + W^yy s_m^y ],  h_n^z = sum_m W^zz s_m^z      */
/*   rho_nm = ((x_m - x_n) mod L, (y_m - y_n) mod L), every m INCLUDING m = n  */
/*   (W(0) is the self-image term).  Every site of the cell exactly once (R3). */
/* colour: -1 = all targets; 0/1 = only targets with (x+y) mod 2 == colour,    */
/* other entries of h are left untouched.                                      */
/* ------------------------------------------------------------------------- */
static void field_at(int L, const double *W, const double *s /* [3][L][L] */, int xn, int yn,
                     double hout[3])
{
    size_t N = (size_t)L * L;
    double hx = 0, hy = 0, hz = 0;
    for (int ym = 0; ym < L; ++ym) {
        for (int xm = 0; xm < L; ++xm) {
            int rx = ((xm - xn) % L + L) % L;
            int ry = ((ym - yn) % L + L) % L;
            size_t w = (size_t)ry * L + rx, m = (size_t)ym * L + xm;
            double sx = s[0 * N + m], sy = s[1 * N + m], sz = s[2 * N + m];
            hx += W[0 * N + w] * sx + W[1 * N + w] * sy;
            hy += W[1 * N + w] * sx + W[2 * N + w] * sy;
            hz += W[3 * N + w] * sz;
        }
    }
    hout[0] = hx;
    hout[1] = hy;
    hout[2] = hz;
}

int oracle_dipole_field(int L, int R, const double *W, const double *s, int colour, double *h)
{
    if (L < 1 || R < 1 || !W || !s || !h || colour < -1 || colour > 1) return -1;
    size_t N = (size_t)L * L;
    long total = (long)R * L * L;
#pragma omp parallel for schedule(static)
    for (long idx = 0; idx < total; ++idx) {
        int r = (int)(idx / (long)N);
        int n = (int)(idx % (long)N);
        int xn = n % L, yn = n / L;
        if (colour >= 0 && ((xn + yn) & 1) != colour) continue;
        double hv[3];
        field_at(L, W, s + (size_t)r * 3 * N, xn, yn, hv);
        for (int c = 0; c < 3; ++c) h[((size_t)r * 3 + c) * N + n] = hv[c];
    }
    return 0;
}

/* field of ONE replica at a list of target sites (for sampled checks at L = 256
 * and for the bounded cpu_baseline sample): h_out[i][3]                         */
int oracle_dipole_field_sampled(int L, const double *W, const double *s /* [3][L][L] */,
                                int ntargets, const int *targets, double *h_out)
{
    if (L < 1 || !W || !s || !targets || !h_out || ntargets < 0) return -1;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < ntargets; ++i) {
        int n = targets[i];
        field_at(L, W, s, n % L, n / L, h_out + 3 * (size_t)i);
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O3. Energy (eq. 11, with the sign reading R7 and R8):        */
/*   E = -J sum_n s_n.(s_{n+x} + s_{n+y})      each NN bond once               */
/*       - sum_n (K2 s_nz^2 + K4 s_nz^4)       eq. 12 as -K2 s_z^2 - K4 s_z^4  */
/*       + (g/2) sum_n s_n . h_n               eq. 1 with images, eq. 2        */
/* out[r] = total energy (not per spin) of replica r; parts[r][3] optional     */
/* (exchange, anisotropy, dipole).                                             */
/* ------------------------------------------------------------------------- */
/* eq. 11 with the dipole field h[R][3][N] of the state s handed in (h = O2 of s): the form the long-run
 * harness uses with a field it evaluated itself (SURVEY.md 8c-O2 allows an fp64 FFT there).     */
int oracle_energy_given_field(int L, int R, double J, double g, const double *K2, const double *K4,
                              const double *s, const double *h, double *out, double *parts)
{
    if (L < 1 || R < 1 || !K2 || !K4 || !s || !h || !out) return -1;
    size_t N = (size_t)L * L;
    for (int r = 0; r < R; ++r) {
        const double *sr = s + (size_t)r * 3 * N, *hr = h + (size_t)r * 3 * N;
        double ex = 0, an = 0, dip = 0;
        for (int y = 0; y < L; ++y) {
            for (int x = 0; x < L; ++x) {
                size_t n = (size_t)y * L + x;
                size_t nx = (size_t)y * L + (x + 1) % L;
                size_t ny = (size_t)((y + 1) % L) * L + x;
                double sx = sr[n], sy = sr[N + n], sz = sr[2 * N + n];
                ex += sx * (sr[nx] + sr[ny]) + sy * (sr[N + nx] + sr[N + ny]) +
                      sz * (sr[2 * N + nx] + sr[2 * N + ny]);
                an += K2[r] * sz * sz + K4[r] * sz * sz * sz * sz;
                dip += sx * hr[n] + sy * hr[N + n] + sz * hr[2 * N + n];
            }
        }
        out[r] = -J * ex - an + 0.5 * g * dip;
        if (parts) {
            parts[3 * r + 0] = -J * ex;
            parts[3 * r + 1] = -an;
            parts[3 * r + 2] = 0.5 * g * dip;
        }
    }
    return 0;
}

int oracle_energy(int L, int R, double J, double g, const double *K2, const double *K4,
                  const double *W, const double *s, double *out, double *parts)
{
    if (L < 1 || R < 1 || !K2 || !K4 || !W || !s || !out) return -1;
    size_t N = (size_t)L * L;
    double *h = (double *)malloc(sizeof(double) * (size_t)R * 3 * N);
    if (!h) return -2;
    oracle_dipole_field(L, R, W, s, -1, h);
    int rc = oracle_energy_given_field(L, R, J, g, K2, K4, s, h, out, parts);
    free(h);
    return rc;
}

/* ------------------------------------------------------------------------- */
/* O4. Random numbers: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11):     */
/* 10 rounds of  (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,                        */
/*   c <- (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0),  key bumped by Weyl        */
/* constants between rounds.  BASELINE.json: "Philox4x32-10 counter-based      */
/* randoms keyed by (seed, replica, step, site)".                              */
/* ------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0;
        k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Keying (R9): key = (seed_lo, seed_hi);
 * counter = (site n = y*L+x, replica r, step_lo, step_hi | tag<<31),
 * tag 0 = half-sweep trial, tag 1 = initial spins.                            */
static void draw(uint64_t seed, uint32_t site, uint32_t replica, uint64_t step, uint32_t tag,
                 uint32_t x[4])
{
    uint32_t ctr[4], key[2];
    ctr[0] = site;
    ctr[1] = replica;
    ctr[2] = (uint32_t)(step & 0xFFFFFFFFu);
    ctr[3] = ((uint32_t)(step >> 32) & 0x7FFFFFFFu) | (tag << 31);
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
    key[1] = (uint32_t)(seed >> 32);
    oracle_philox4x32_10(ctr, key, x);
}

/* 32 random bits -> u = (2 (x >> 9) + 1) 2^-24: an odd multiple of 2^-24, strictly
 * inside (0,1), exactly representable in fp32 and fp64 (R9).                   */
static double to_unit(uint32_t x)
{
    return (double)(2u * (x >> 9) + 1u) * (1.0 / 16777216.0);
}

/* Uniform point on S^2 (App. A: one angle uniform on [0, 2pi],
 * the other arccos of a uniform on [-1, 1]; reading R10): z = 2 u0 - 1,
 * phi = 2 pi u1, s' = (sqrt(1 - z^2) cos phi, sqrt(1 - z^2) sin phi, z).         */
static void sphere_point(uint32_t x0, uint32_t x1, double sp[3])
{
    double z = 2.0 * to_unit(x0) - 1.0;
    double phi = 2.0 * ORACLE_PI * to_unit(x1);
    double rho = sqrt((1.0 - z) * (1.0 + z));
    sp[0] = rho * cos(phi);
    sp[1] = rho * sin(phi);
    sp[2] = z;
}

/* expose the draw for tests: out = {s'_x, s'_y, s'_z, u} and the raw words */
void oracle_trial_draw(uint64_t seed, uint32_t site, uint32_t replica, uint64_t step, uint32_t tag,
                       double out[4], uint32_t raw[4])
{
    uint32_t x[4];
    draw(seed, site, replica, step, tag, x);
    sphere_point(x[0], x[1], out);
    out[3] = to_unit(x[2]);
    if (raw) memcpy(raw, x, sizeof(x));
}

/* a4. initial spins: mode 0 = uniform on S^2 from (seed, replica, site) with tag 1,
 * mode 1 = all +z (BASELINE.json configs).                                     */
int oracle_init_spins(int L, int R, int mode, uint64_t seed, double *s)
{
    if (L < 1 || R < 1 || !s || mode < 0 || mode > 1) return -1;
    size_t N = (size_t)L * L;
    for (int r = 0; r < R; ++r) {
        for (size_t n = 0; n < N; ++n) {
            double sp[3] = {0.0, 0.0, 1.0};
            if (mode == 0) {
                uint32_t x[4];
                draw(seed, (uint32_t)n, (uint32_t)r, 0, 1u, x);
                sphere_point(x[0], x[1], sp);
            }
            for (int c = 0; c < 3; ++c) s[((size_t)r * 3 + c) * N + n] = sp[c];
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O5. Energy difference of a single-spin trial and the Metropolis half-sweep */
/* ------------------------------------------------------------------------- */

/* dE for replacing s_n by s' with every other spin fixed, given the dipole field
 * h_n of the CURRENT state (which contains the self term W(0) s_n):
 *   delta = s' - s_n
 *   dE = -J delta.(s_{n+x} + s_{n-x} + s_{n+y} + s_{n-y})          (eq. 11, exchange)
 *        - K2 (s'_z^2 - s_z^2) - K4 (s'_z^4 - s_z^4)                (eq. 12)
 *        + g [ delta.h_n + (1/2) delta.W(0).delta ]                 (eq. 1-2)
 * The last term: E_dip = (g/2) sum_{n,m} s_n W(rho_nm) s_m is quadratic in s_n, the
 * cross terms give delta.h_n and the m = n term gives (1/2) delta.W(0).delta
 * (R12: the trial spin is coupled to its own images exactly).  W^xy(0) = 0 and
 * W^xx(0) = W^yy(0) by the square symmetry, but the general form is kept.        */
double oracle_delta_e(int L, double J, double g, double K2, double K4, const double *W,
                      const double *s /* [3][L][L] */, const double h_n[3], int n,
                      const double sp[3])
{
    size_t N = (size_t)L * L;
    int x = n % L, y = n / L;
    size_t e = (size_t)y * L + (x + 1) % L, w = (size_t)y * L + (x + L - 1) % L;
    size_t no = (size_t)((y + 1) % L) * L + x, so = (size_t)((y + L - 1) % L) * L + x;
    double sx = s[n], sy = s[N + n], sz = s[2 * N + n];
    double d[3] = {sp[0] - sx, sp[1] - sy, sp[2] - sz};
    double nb[3];
    for (int c = 0; c < 3; ++c) nb[c] = s[c * N + e] + s[c * N + w] + s[c * N + no] + s[c * N + so];
    double dE_ex = -J * (d[0] * nb[0] + d[1] * nb[1] + d[2] * nb[2]);
    double dE_an = -K2 * (sp[2] * sp[2] - sz * sz) -
                   K4 * (sp[2] * sp[2] * sp[2] * sp[2] - sz * sz * sz * sz);
    double w0xx = W[0 * N], w0xy = W[1 * N], w0yy = W[2 * N], w0zz = W[3 * N];
    double self = 0.5 * (d[0] * (w0xx * d[0] + w0xy * d[1]) + d[1] * (w0xy * d[0] + w0yy * d[1]) +
                         d[2] * w0zz * d[2]);
    double dE_dip = g * (d[0] * h_n[0] + d[1] * h_n[1] + d[2] * h_n[2] + self);
    return dE_ex + dE_an + dE_dip;
}

/* One checkerboard half-sweep (BASELINE.json north_star; eq. 7,
 * :98, :102-118 "simultaneous flipping" approximation H3 - H1 ~ H2 - H0):
 *   c = step & 1; active sites (x + y) mod 2 == c                      (R11)
 *   (i)  h <- O2 from the state AT ENTRY, all sources of both colours   (R13)
 *   (ii) for every active site n and replica r, independently:
 *        (s', u) from Philox(seed; n, r, step); dE as above with the frozen h;
 *        margin = dE/T_r + ln u;  accept  <=>  margin < 0               (eq. 7, R14)
 *        accepted sites take s' (replaced, never incremented).
 * The exchange neighbours of an active site all have the other colour, so the
 * exchange part is exact; only the dipole part sees "old" spins of the other
 * simultaneously updated sites.
 * Outputs (each nullable): h_out [R][3][N] (active sites written), accept_out
 * [R][N] bytes (active sites written, 0/1), margin_out [R][N], trial_out [R][3][N]. */
int oracle_halfsweep_given_field(int L, int R, double J, double g, const double *K2, const double *K4,
                                 const double *W, double *s, const double *T, uint64_t seed,
                                 uint64_t step, const double *h, double *h_out, uint8_t *accept_out,
                                 double *margin_out, double *trial_out);

int oracle_halfsweep(int L, int R, double J, double g, const double *K2, const double *K4,
                     const double *W, double *s, const double *T, uint64_t seed, uint64_t step,
                     double *h_out, uint8_t *accept_out, double *margin_out, double *trial_out)
{
    if (L < 2 || (L & 1) || R < 1 || !K2 || !K4 || !W || !s || !T) return -1;
    for (int r = 0; r < R; ++r)
        if (!(T[r] > 0.0)) return -1;
    size_t N = (size_t)L * L;
    int colour = (int)(step & 1u);
    double *h = (double *)malloc(sizeof(double) * (size_t)R * 3 * N);
    if (!h) return -2;
    memset(h, 0, sizeof(double) * (size_t)R * 3 * N);
    oracle_dipole_field(L, R, W, s, colour, h);             /* (i): O2 on the state at entry */
    int rc = oracle_halfsweep_given_field(L, R, J, g, K2, K4, W, s, T, seed, step, h, h_out,
                                          accept_out, margin_out, trial_out);
    free(h);
    return rc;
}

/* Step (ii) of the half-sweep alone, with the frozen field h[R][3][N] of the state at entry handed in
 * (only its entries at active sites are read).  oracle_halfsweep is "h <- O2, then this".  The long-run
 * harness calls it with a field it evaluated by fp64 FFT (allowed in the harness to make
 * long oracle runs affordable; tests pin that field to O2 first); W is still needed for W(0).    */
int oracle_halfsweep_given_field(int L, int R, double J, double g, const double *K2, const double *K4,
                                 const double *W, double *s, const double *T, uint64_t seed,
                                 uint64_t step, const double *h, double *h_out, uint8_t *accept_out,
                                 double *margin_out, double *trial_out)
{
    if (L < 2 || (L & 1) || R < 1 || !K2 || !K4 || !W || !s || !T || !h) return -1;
    for (int r = 0; r < R; ++r)
        if (!(T[r] > 0.0)) return -1;
    size_t N = (size_t)L * L;
    int colour = (int)(step & 1u);
    double *snew = (double *)malloc(sizeof(double) * (size_t)R * 3 * N);
    if (!snew) return -2;
    memcpy(snew, s, sizeof(double) * (size_t)R * 3 * N);
    long total = (long)R * (long)N;
#pragma omp parallel for schedule(static)
    for (long idx = 0; idx < total; ++idx) {
        int r = (int)(idx / (long)N);
        int n = (int)(idx % (long)N);
        int x = n % L, y = n / L;
        if (((x + y) & 1) != colour) continue;
        const double *sr = s + (size_t)r * 3 * N; /* state at entry */
        uint32_t rnd[4];
        double sp[3];
        draw(seed, (uint32_t)n, (uint32_t)r, step, 0u, rnd);
        sphere_point(rnd[0], rnd[1], sp);
        double u = to_unit(rnd[2]);
        double hn[3] = {h[((size_t)r * 3 + 0) * N + n], h[((size_t)r * 3 + 1) * N + n],
                        h[((size_t)r * 3 + 2) * N + n]};
        double dE = oracle_delta_e(L, J, g, K2[r], K4[r], W, sr, hn, n, sp);
        double margin = dE / T[r] + log(u);
        int acc = margin < 0.0;
        if (acc)
            for (int c = 0; c < 3; ++c) snew[((size_t)r * 3 + c) * N + n] = sp[c];
        if (accept_out) accept_out[(size_t)r * N + n] = (uint8_t)acc;
        if (margin_out) margin_out[(size_t)r * N + n] = margin;
        if (trial_out)
            for (int c = 0; c < 3; ++c) trial_out[((size_t)r * 3 + c) * N + n] = sp[c];
        if (h_out)
            for (int c = 0; c < 3; ++c) h_out[((size_t)r * 3 + c) * N + n] = hn[c];
    }
    memcpy(s, snew, sizeof(double) * (size_t)R * 3 * N);
    free(snew);
    return 0;
}

/* Exact sequential single-spin Metropolis over the same sites, in site order,
 * with the same random numbers but the field recomputed after every accepted
 * move (no approximation).  Used only by tests that measure what the frozen-field
 * approximation changes (eq. 8); O(N^2) per site, tiny L only.
 * margin_out (nullable, [R][N], active sites written) = dE/T + ln u as each site saw it.
 * Pin at g != 0 (tests/test_oracle_physics.py::test_eq8_sequential_minus_frozen_halfsweep):
 * with every move accepted, margin_seq(k) - margin_frozen(k) = (g/T) sum_{j<k} delta_j.W(rho_jk).delta_k. */
int oracle_halfsweep_sequential(int L, int R, double J, double g, const double *K2,
                                const double *K4, const double *W, double *s, const double *T,
                                uint64_t seed, uint64_t step, uint8_t *accept_out, double *margin_out)
{
    if (L < 2 || (L & 1) || R < 1 || !K2 || !K4 || !W || !s || !T) return -1;
    size_t N = (size_t)L * L;
    int colour = (int)(step & 1u);
    for (int r = 0; r < R; ++r) {
        double *sr = s + (size_t)r * 3 * N;
        for (int n = 0; n < (int)N; ++n) {
            int x = n % L, y = n / L;
            if (((x + y) & 1) != colour) continue;
            uint32_t rnd[4];
            double sp[3], hn[3];
            draw(seed, (uint32_t)n, (uint32_t)r, step, 0u, rnd);
            sphere_point(rnd[0], rnd[1], sp);
            double u = to_unit(rnd[2]);
            field_at(L, W, sr, x, y, hn);
            double dE = oracle_delta_e(L, J, g, K2[r], K4[r], W, sr, hn, n, sp);
            double margin = dE / T[r] + log(u);
            int acc = margin < 0.0;
            if (acc)
                for (int c = 0; c < 3; ++c) sr[c * N + n] = sp[c];
            if (accept_out) accept_out[(size_t)r * N + n] = (uint8_t)acc;
            if (margin_out) margin_out[(size_t)r * N + n] = margin;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O6. Observables per replica: out[r] = { E/N, m_z, M_par, eta }             */
/*   E/N   : O3 / N                                           (eq. 11)         */
/*   m_z   : N^-1 sum_i s_i^z                                 (BASELINE.json)   */
/*   M_par : (M_x^2 + M_y^2)^(1/2), M_a = N^-1 sum_i s_i^a    (eq. 16, :225)    */
/*   eta   : (2/pi) ( N^-1 sum_i (theta_i - pi/2)^2 )^(1/2),                    */
/*           theta_i = arccos s_i^z   (eq. 17, :232, per-snapshot reading R15)  */
/* ------------------------------------------------------------------------- */
static void magnetisation_and_cone(int L, const double *sr, double out[3])
{
    size_t N = (size_t)L * L;
    double mx = 0, my = 0, mz = 0, q = 0;
    for (size_t n = 0; n < N; ++n) {
        mx += sr[n];
        my += sr[N + n];
        mz += sr[2 * N + n];
        double cz = sr[2 * N + n];
        if (cz > 1.0) cz = 1.0;
        if (cz < -1.0) cz = -1.0;
        double th = acos(cz) - 0.5 * ORACLE_PI;
        q += th * th;
    }
    mx /= (double)N; my /= (double)N; mz /= (double)N; q /= (double)N;
    out[0] = mz;
    out[1] = sqrt(mx * mx + my * my);
    out[2] = (2.0 / ORACLE_PI) * sqrt(q);
}

int oracle_observables(int L, int R, double J, double g, const double *K2, const double *K4,
                       const double *W, const double *s, double *out)
{
    if (L < 1 || R < 1 || !s || !out) return -1;
    size_t N = (size_t)L * L;
    double *E = (double *)malloc(sizeof(double) * R);
    if (!E) return -2;
    int rc = oracle_energy(L, R, J, g, K2, K4, W, s, E, NULL);
    if (rc) { free(E); return rc; }
    for (int r = 0; r < R; ++r) {
        out[4 * r + 0] = E[r] / (double)N;
        magnetisation_and_cone(L, s + (size_t)r * 3 * N, out + 4 * r + 1);
    }
    free(E);
    return 0;
}

/* the same with the field h = O2 of s handed in (see oracle_energy_given_field) */
int oracle_observables_given_field(int L, int R, double J, double g, const double *K2,
                                   const double *K4, const double *s, const double *h, double *out)
{
    if (L < 1 || R < 1 || !s || !h || !out) return -1;
    size_t N = (size_t)L * L;
    double *E = (double *)malloc(sizeof(double) * R);
    if (!E) return -2;
    int rc = oracle_energy_given_field(L, R, J, g, K2, K4, s, h, E, NULL);
    if (rc) { free(E); return rc; }
    for (int r = 0; r < R; ++r) {
        out[4 * r + 0] = E[r] / (double)N;
        magnetisation_and_cone(L, s + (size_t)r * 3 * N, out + 4 * r + 1);
    }
    free(E);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O7. Domain-wall counts (eq. 14) per replica and component */
/*   n_v^a = sum_i [ 1 - sgn(s_i^a s_{i+y}^a) ],  n_h^a = sum_i [ 1 - sgn(s_i^a s_{i+x}^a) ]  */
/* with periodic neighbours i+x = ((x+1) mod L, y), i+y = (x, (y+1) mod L), every  */
/* bond once.  sgn(a b) is taken as sgn(a) sgn(b) (the same number, and immune to   */
/* the product underflowing), sgn(0) = 0, so every term is 0, 1 or 2 and the sums   */
/* are integers.  out[r] = { n_h^x, n_v^x, n_h^y, n_v^y, n_h^z, n_v^z }.             */
/* Derived per snapshot (the thermal averages of eq. 15 and the variances of       */
/* eq. 18 are statistics the caller takes over snapshots):                         */
/*   wall density  (n_v^z + n_h^z) / (4N)        */
/*   O_a = |n_h^a - n_v^a| / (n_h^a + n_v^a)                 (eq. 15, :207);       */
/*         0 when there is no wall at all (paper silent; R20)            */
/* ------------------------------------------------------------------------- */
static int oracle_sgn(double v) { return (v > 0.0) - (v < 0.0); }

int oracle_wall_counts(int L, int R, const double *s, long long *out)
{
    if (L < 1 || R < 1 || !s || !out) return -1;
    size_t N = (size_t)L * L;
    for (int r = 0; r < R; ++r) {
        for (int c = 0; c < 3; ++c) {
            const double *f = s + ((size_t)r * 3 + c) * N;
            long long nh = 0, nv = 0;
            for (int y = 0; y < L; ++y) {
                for (int x = 0; x < L; ++x) {
                    int si = oracle_sgn(f[(size_t)y * L + x]);
                    int sx = oracle_sgn(f[(size_t)y * L + (x + 1) % L]);
                    int sy = oracle_sgn(f[(size_t)((y + 1) % L) * L + x]);
                    nh += 1 - si * sx;
                    nv += 1 - si * sy;
                }
            }
            out[6 * r + 2 * c + 0] = nh;
            out[6 * r + 2 * c + 1] = nv;
        }
    }
    return 0;
}

/* derived[r] = { wall density, O_x, O_y, O_z } from the counts of oracle_wall_counts */
int oracle_wall_order(int L, int R, const long long *counts, double *derived)
{
    if (L < 1 || R < 1 || !counts || !derived) return -1;
    double N = (double)L * (double)L;
    for (int r = 0; r < R; ++r) {
        const long long *n = counts + 6 * r;
        derived[4 * r + 0] = (double)(n[4] + n[5]) / (4.0 * N);
        for (int c = 0; c < 3; ++c) {
            long long nh = n[2 * c], nv = n[2 * c + 1];
            long long d = nh > nv ? nh - nv : nv - nh;
            derived[4 * r + 1 + c] = (nh + nv) > 0 ? (double)d / (double)(nh + nv) : 0.0;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O8. The paper's own update schedule (section 3.1; App. A :307-361) */
/* One pass p of the algorithm with stride l (l >= 2, l | L):                     */
/*   (i)   a site i_1 = (S_1, S_2) is selected at random, S_1, S_2 in [0, l)       */
/*         (App. A "S_1 = Random Integer in [1, l]", 0-based here; reading R21:    */
/*         words x0, x1 of Philox(seed; 0xFFFFFFFF, 0xFFFFFFFF, p), S = x mod l);  */
/*   (ii)  update sites i = (a l, b l) + i_1, a, b in [0, L/l): n = (L/l)^2 sites   */
/*         (the "a, b in [0, L/l]" and "T_id <= L^2 \ l^2" of the text count one    */
/*         too many: R3/A19 reading, every site of the sub-lattice exactly once);   */
/*   (iii) for each update site and replica a trial spin and u from                 */
/*         Philox(seed; site, replica, step = p) as in O5; flip != 0 selects the    */
/*         Ising move of App. B (:366) instead: the trial is the reversed spin;     */
/*   (iv)  dipole energies of all n sites from the state AT ENTRY to the pass       */
/*         ("simultaneous flipping", :102-118), exchange and anisotropy exact       */
/*         (update sites are never nearest neighbours for l >= 2);                  */
/*   (v)   accept <=> dE/T + ln u < 0.                                              */
/* sequential != 0 runs the same sites in order a fastest, with the same random     */
/* numbers, recomputing the field from the CURRENT state for every site: the        */
/* conventional Metropolis the paper compares against (App. B).                     */
/* offset_out[2] (nullable) = {S_1, S_2}; accept_out [R][N], margin_out [R][N],     */
/* trial_out [R][3][N] (nullable) are written at the update sites only.             */
/* ------------------------------------------------------------------------- */
void oracle_sublattice_offset(uint64_t seed, uint64_t pass, int l, int offset[2])
{
    uint32_t ctr[4], key[2], x[4];
    ctr[0] = 0xFFFFFFFFu;
    ctr[1] = 0xFFFFFFFFu;
    ctr[2] = (uint32_t)(pass & 0xFFFFFFFFu);
    ctr[3] = (uint32_t)(pass >> 32) & 0x7FFFFFFFu;
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
    key[1] = (uint32_t)(seed >> 32);
    oracle_philox4x32_10(ctr, key, x);
    offset[0] = (int)(x[0] % (uint32_t)l);
    offset[1] = (int)(x[1] % (uint32_t)l);
}

int oracle_sublattice_pass(int L, int R, double J, double g, const double *K2, const double *K4,
                           const double *W, double *s, const double *T, uint64_t seed,
                           uint64_t pass, int l, int flip, int sequential, int *offset_out,
                           uint8_t *accept_out, double *margin_out, double *trial_out)
{
    if (L < 2 || R < 1 || l < 2 || L % l || !K2 || !K4 || !W || !s || !T) return -1;
    for (int r = 0; r < R; ++r)
        if (!(T[r] > 0.0)) return -1;
    size_t N = (size_t)L * L;
    int nl = L / l, off[2];
    oracle_sublattice_offset(seed, pass, l, off);
    if (offset_out) { offset_out[0] = off[0]; offset_out[1] = off[1]; }
    double *entry = (double *)malloc(sizeof(double) * 3 * N);
    if (!entry) return -2;
    for (int r = 0; r < R; ++r) {
        double *sr = s + (size_t)r * 3 * N;
        memcpy(entry, sr, sizeof(double) * 3 * N);          /* the state at entry to the pass */
        for (int b = 0; b < nl; ++b) {
            for (int a = 0; a < nl; ++a) {
                int x = off[0] + l * a, y = off[1] + l * b;
                int n = y * L + x;
                uint32_t rnd[4];
                double sp[3], hn[3];
                draw(seed, (uint32_t)n, (uint32_t)r, pass, 0u, rnd);
                if (flip) {
                    for (int c = 0; c < 3; ++c) sp[c] = -entry[c * N + n];
                } else {
                    sphere_point(rnd[0], rnd[1], sp);
                }
                double u = to_unit(rnd[2]);
                /* frozen: every site sees the state at entry; sequential: the current one.
                 * The site's own spin and its four neighbours are the same in both (no
                 * other update site touches them), so only the dipole sum differs.       */
                const double *view = sequential ? sr : entry;
                field_at(L, W, view, x, y, hn);
                double dE = oracle_delta_e(L, J, g, K2[r], K4[r], W, view, hn, n, sp);
                double margin = dE / T[r] + log(u);
                int acc = margin < 0.0;
                if (acc)
                    for (int c = 0; c < 3; ++c) sr[c * N + n] = sp[c];
                if (accept_out) accept_out[(size_t)r * N + n] = (uint8_t)acc;
                if (margin_out) margin_out[(size_t)r * N + n] = margin;
                if (trial_out)
                    for (int c = 0; c < 3; ++c) trial_out[((size_t)r * 3 + c) * N + n] = sp[c];
            }
        }
    }
    free(entry);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O9. Staggered magnetisation of App. B (after Binder and Landau [61]) */
/* for stripes of width h = 1: four sub-lattices of the 2 x 2 plaquette,             */
/*   1 = (x even, y even), 2 = (x odd, y even), 3 = (x odd, y odd), 4 = (x even, y odd), */
/*   m_lambda = N^-1 sum_{i in lambda} s_i^z   (so that a perfect stripe state gives 1; */
/*   the paper does not state the normalisation: DESIGN.md R23),                       */
/*   m_h = m_1 + m_2 - m_3 - m_4 (horizontal stripes: rows alternate),                 */
/*   m_v = m_1 + m_4 - m_3 - m_2 (vertical stripes: columns alternate),                */
/*   m_st = (m_h^2 + m_v^2)^(1/2) per snapshot; <m_st> and chi_st are the caller's.     */
/* out[r] = { m_h, m_v, m_st }.                                                        */
/* ------------------------------------------------------------------------- */
int oracle_staggered(int L, int R, const double *s, double *out)
{
    if (L < 2 || (L & 1) || R < 1 || !s || !out) return -1;
    size_t N = (size_t)L * L;
    for (int r = 0; r < R; ++r) {
        const double *sz = s + ((size_t)r * 3 + 2) * N;
        double m[4] = {0, 0, 0, 0};
        for (int y = 0; y < L; ++y) {
            for (int x = 0; x < L; ++x) {
                int lambda = (y & 1) ? ((x & 1) ? 2 : 3) : ((x & 1) ? 1 : 0);
                m[lambda] += sz[(size_t)y * L + x];
            }
        }
        for (int k = 0; k < 4; ++k) m[k] /= (double)N;
        double mh = m[0] + m[1] - m[2] - m[3];
        double mv = m[0] + m[3] - m[2] - m[1];
        out[3 * r + 0] = mh;
        out[3 * r + 1] = mv;
        out[3 * r + 2] = sqrt(mh * mh + mv * mv);
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O10. Ensemble statistics over n recorded states:          */
/*   thermal average <X> = n^-1 sum_t X_t,                                      */
/*   variance sigma^2(X) = <(X - <X>)^2> = <X^2> - <X>^2          (eq. 18, :265) */
/*   standard error SE = ((<X^2> - <X>^2) / n)^(1/2)              (eq. 13, :177) */
/* x[t][k], t < n snapshots, k < K quantities; outputs mean[K], var[K], se[K].  */
/* ------------------------------------------------------------------------- */
int oracle_ensemble(int n, int K, const double *x, double *mean, double *var, double *se)
{
    if (n < 1 || K < 1 || !x || !mean || !var || !se) return -1;
    for (int k = 0; k < K; ++k) {
        double m = 0.0;
        for (int t = 0; t < n; ++t) m += x[(size_t)t * K + k];
        m /= (double)n;
        double v = 0.0;
        for (int t = 0; t < n; ++t) {
            double d = x[(size_t)t * K + k] - m;
            v += d * d;
        }
        v /= (double)n;
        mean[k] = m;
        var[k] = v;
        se[k] = sqrt(v / (double)n);
    }
    return 0;
}
