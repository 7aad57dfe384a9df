/*
 * oracle/xy_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU statement of the Swendsen-Wang multi-cluster
 * sweep of the 2D classical XY model with Wolff's embedded-cluster projection,
 * its observables and the helicity-modulus PCC driver, as used in
 * arXiv 1210.6116 (Komura & Okabe).  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build or call this file.
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_1210_6116_b200/csrc/ and must never be imported by it.
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fno-fast-math -shared -fPIC
 *        (see oracle/build.py).  -ffp-contract=off: every fp64 operation below
 *        is one IEEE-754 round-to-nearest operation, in the order written.
 *
 * What the paper fixes and what it does not (citations are PAPER.md lines):
 *   - Hamiltonian  H = -J sum_<ij> cos(theta_i - theta_j), LxL periodic, J=1
 *     (PAPER.md:38-42 Eq. 3; :66 "unit of J=1").
 *   - helicity modulus  Y = <e> - (J L^2/T) <s^2>,  e,s = (1/L^2) sum over the
 *     links of ONE direction of cos, sin(theta_i - theta_j)
 *     (Eq. 4-6; Eq. 5's subscript "c" is extraction damage for
 *     "x", see the sentence at :54).
 *   - <m^2> = chi/L^2, chi(0) = (1/N)|sum_r s(r)|^2 (PAPER.md:107 Eq. 9, :119
 *     Eq. 10).
 *   - PCC rule: if beta*Y < 0.636508 raise beta by dbeta, else lower it
 *     (PAPER.md:62); Y measured over 1000 MCS, dbeta = 0.0005, 60000 MCS
 *     discarded.
 *   - The update itself is only named (Swendsen-Wang :22, Wolff's embedded
 *     cluster formalism :26); its formulas are the textbook ones fixed by
 *     BASELINE.json's north_star and listed as readings in DESIGN.md section 3:
 *     random unit vector r=(cos phi, sin phi) per sweep; sigma_i = s_i . r;
 *     bond <ij> active with probability 1-exp(-2 beta sigma_i sigma_j) when
 *     sigma_i sigma_j > 0; every cluster reflected s -> s - 2(s.r)r with
 *     probability 1/2.
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   philox      : cuRAND's host Philox4_32_10 generator (independent library);
 *                 bijectivity / distinctness; uniform moments.
 *   bonds       : closed-form densities and exact special cases.
 *   label       : scipy.sparse.csgraph.connected_components and a BFS written
 *                 in the test; exhaustive enumeration of all bond sets L<=3.
 *   flip        : reflection identities; involution.
 *   sweep       : exact detailed balance + stationarity of the 2x2 transition
 *                 matrix; 4x4 Ising limit vs exact enumeration; beta->0; low-T
 *                 spin wave; the paper's Table I row L=64.
 *   observe     : independent numpy evaluation with math.fsum.
 *   pcc         : injected monotone observable; paper's beta_KT(64).
 *   fourier     : numpy FFT of the spin field; plane wave and uniform closed forms;
 *                 Eq. 8 inverts the Ornstein-Zernike form exactly; xi_2nd/L of the
 *                 paper's Table I row L=64.
 *   potts       : (section at the end of this file; tests/test_oracle_potts.py) exact one-step transition
 *                 matrix and Boltzmann weights of the 2x2 torus (q = 3), enumeration of all 2^16 states
 *                 of the 4x4 q = 2 model, bond-rule closed forms, uniformity and independence of the
 *                 fresh spins, e(beta_c) = -(1 + 1/sqrt q) at the self-dual point.
 * No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define XYO_TWO_PI 6.283185307179586  /* 0x401921FB54442D18, fl64(2 pi) */
#define XYO_PI     3.141592653589793  /* 0x400921FB54442D18, fl64(pi)   */

enum { XYO_TAG_INIT = 0, XYO_TAG_DIR = 1, XYO_TAG_BOND = 2, XYO_TAG_FLIP = 3, XYO_TAG_BOND_LO = 4 };

/* ------------------------------------------------------------------------- */
/* O1. RNG: Philox4x32 with 10 rounds (Salmon, Moraes, Dror, Shaw, SC'11).     */
/* The paper is silent on the RNG; north_star mandates a counter-based Philox */
/* keyed by (seed, sweep, site/bond).                                          */
/* ------------------------------------------------------------------------- */
void xyo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   /* multipliers  */
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   /* Weyl key bumps */
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
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* key = (seed lo, seed hi); counter = (idx lo, idx hi, (u32)t, tag). */
void xyo_rng(uint64_t seed, uint64_t idx, uint64_t t, uint32_t tag, uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)(idx & 0xffffffffu), (uint32_t)(idx >> 32),
                        (uint32_t)t, tag };
    xyo_philox4x32_10(ctr, key, out);
}

/* U(w) = (w + 0.5) * 2^-32, exact in fp64, strictly inside (0,1). */
double xyo_uniform(uint32_t w)
{
    return ((double)w + 0.5) * (1.0 / 4294967296.0);
}

/* ------------------------------------------------------------------------- */
/* O2. Initial state.  init = 0 cold (all theta = +0.0f); 1 hot.               */
/* hot: theta_i = (float)(2pi * (w0>>8) * 2^-24), w = rng(seed, i, 0, INIT).   */
/* ------------------------------------------------------------------------- */
int xyo_init(float *theta, uint32_t L, uint64_t seed, int init)
{
    uint64_t N = (uint64_t)L * L;
    if (init == 0) {
        for (uint64_t i = 0; i < N; ++i) theta[i] = 0.0f;
        return 0;
    }
    if (init != 1) return -1;
    for (uint64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        xyo_rng(seed, i, 0, XYO_TAG_INIT, w);
        double frac = (double)(w[0] >> 8) * (1.0 / 16777216.0);
        theta[i] = (float)(XYO_TWO_PI * frac);
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O3. Direction of the sweep: phi uniform on [0, 2pi), r = (cos phi, sin phi) */
/* (Wolff embedding; one r per sweep, north_star).               */
/* ------------------------------------------------------------------------- */
double xyo_phi(uint64_t seed, uint64_t t)
{
    uint32_t w[4];
    xyo_rng(seed, 0, t, XYO_TAG_DIR, w);
    return XYO_TWO_PI * ((double)w[0] * (1.0 / 4294967296.0));
}

/* ------------------------------------------------------------------------- */
/* O4. Bonds.  sigma_i = s_i . r = cos(theta_i - phi); a bond <ij> is active   */
/* iff u < p, p = 1 - exp(-2 beta sigma_i sigma_j) = -expm1(-2 beta a).        */
/* For a <= 0, p <= 0 < u: the "sigma_i sigma_j > 0" condition is implied.     */
/* ------------------------------------------------------------------------- */
double xyo_sigma(float theta, double phi)
{
    return cos((double)theta - phi);
}

double xyo_bond_prob(double beta, double sigma_i, double sigma_j)
{
    double a = sigma_i * sigma_j;
    double x = (-2.0 * beta) * a;
    return -expm1(x);
}

/* uniforms of site i at sweep t.  Two Philox calls per QUAD of sites q = i>>2, */
/* A = rng(seed, q, t, BOND) and B = rng(seed, q, t, BOND_LO); site 4q+j takes   */
/* the 32-bit words  wx = (lo16(A_j) << 16) | lo16(B_j)  (x bond) and            */
/* wy = (hi16(A_j) << 16) | hi16(B_j)  (y bond):  call A holds the 16 leading    */
/* bits of all 8 uniforms of the quad, call B the 16 trailing bits.              */
void xyo_bond_uniforms_site(uint64_t seed, uint64_t t, uint64_t i, double *ux, double *uy)
{
    uint32_t A[4], B[4];
    unsigned j = (unsigned)(i & 3u);
    xyo_rng(seed, i >> 2, t, XYO_TAG_BOND, A);
    xyo_rng(seed, i >> 2, t, XYO_TAG_BOND_LO, B);
    *ux = xyo_uniform(((A[j] & 0xffffu) << 16) | (B[j] & 0xffffu));
    *uy = xyo_uniform((A[j] & 0xffff0000u) | (B[j] >> 16));
}

static uint64_t right_of(uint64_t x, uint64_t y, uint64_t L) { return y * L + ((x + 1) % L); }
static uint64_t down_of (uint64_t x, uint64_t y, uint64_t L) { return ((y + 1) % L) * L + x; }

/* bonds[i] = bx(i) | by(i) << 1.  bx(i): bond (x,y)-(x+1 mod L, y);
 * by(i): bond (x,y)-(x, y+1 mod L).  ux, uy: the 2N uniforms, injected.
 * margin_x / margin_y (optional, may be NULL): m = u - p of every bond.      */
void xyo_bonds_from_u(const float *theta, uint32_t L32, double beta, double phi,
                      const double *ux, const double *uy, uint8_t *bonds,
                      double *margin_x, double *margin_y)
{
    uint64_t L = L32;
    for (uint64_t y = 0; y < L; ++y) {
        for (uint64_t x = 0; x < L; ++x) {
            uint64_t i = y * L + x;
            double si = xyo_sigma(theta[i], phi);
            double px = xyo_bond_prob(beta, si, xyo_sigma(theta[right_of(x, y, L)], phi));
            double py = xyo_bond_prob(beta, si, xyo_sigma(theta[down_of(x, y, L)], phi));
            uint8_t b = 0;
            if (ux[i] < px) b |= 1u;
            if (uy[i] < py) b |= 2u;
            bonds[i] = b;
            if (margin_x) margin_x[i] = ux[i] - px;
            if (margin_y) margin_y[i] = uy[i] - py;
        }
    }
}

/* Same, drawing the uniforms from the RNG on the fly (no 2N-double arrays).   */
void xyo_bonds(const float *theta, uint32_t L32, double beta, double phi,
               uint64_t seed, uint64_t t, uint8_t *bonds,
               double *margin_x, double *margin_y)
{
    uint64_t L = L32;
    for (uint64_t y = 0; y < L; ++y) {
        for (uint64_t x = 0; x < L; ++x) {
            uint64_t i = y * L + x;
            double ux, uy;
            xyo_bond_uniforms_site(seed, t, i, &ux, &uy);
            double si = xyo_sigma(theta[i], phi);
            double px = xyo_bond_prob(beta, si, xyo_sigma(theta[right_of(x, y, L)], phi));
            double py = xyo_bond_prob(beta, si, xyo_sigma(theta[down_of(x, y, L)], phi));
            uint8_t b = 0;
            if (ux < px) b |= 1u;
            if (uy < py) b |= 2u;
            bonds[i] = b;
            if (margin_x) margin_x[i] = ux - px;
            if (margin_y) margin_y[i] = uy - py;
        }
    }
}

/* margin m = u - p of one bond (dir 0: x, 1: y) -- for the parity report.     */
double xyo_bond_margin(const float *theta, uint32_t L32, double beta, double phi,
                       uint64_t seed, uint64_t t, uint64_t i, int dir)
{
    uint64_t L = L32, x = i % L, y = i / L;
    double ux, uy;
    xyo_bond_uniforms_site(seed, t, i, &ux, &uy);
    uint64_t j = dir == 0 ? right_of(x, y, L) : down_of(x, y, L);
    double p = xyo_bond_prob(beta, xyo_sigma(theta[i], phi), xyo_sigma(theta[j], phi));
    return (dir == 0 ? ux : uy) - p;
}

/* ------------------------------------------------------------------------- */
/* O5. Cluster labels: sequential union-find, the smaller index becomes the    */
/* root, so label[i] = minimum site index of i's connected component.          */
/* (Cluster labeling is the step the paper names at PAPER.md:30-34; the        */
/* canonical minimum-index label is the fixed point of the label-equivalence   */
/* methods cited there.)  Parents are held as u32 (N <= 2^32).                 */
/* Returns the number of clusters, or (uint64_t)-1 on allocation failure.      */
/* ------------------------------------------------------------------------- */
static uint32_t uf_find(uint32_t *parent, uint32_t a)
{
    uint32_t r = a;
    while (parent[r] != r) r = parent[r];
    while (parent[a] != r) { uint32_t nxt = parent[a]; parent[a] = r; a = nxt; }
    return r;
}

static void uf_union(uint32_t *parent, uint32_t a, uint32_t b)
{
    uint32_t ra = uf_find(parent, a), rb = uf_find(parent, b);
    if (ra == rb) return;
    if (ra < rb) parent[rb] = ra; else parent[ra] = rb;
}

uint64_t xyo_label(const uint8_t *bonds, uint32_t L32, int64_t *label)
{
    uint64_t L = L32, N = L * L;
    uint32_t *parent = (uint32_t *)malloc(N * sizeof(uint32_t));
    if (!parent) return (uint64_t)-1;
    for (uint64_t i = 0; i < N; ++i) parent[i] = (uint32_t)i;
    for (uint64_t y = 0; y < L; ++y) {
        for (uint64_t x = 0; x < L; ++x) {
            uint64_t i = y * L + x;
            if (bonds[i] & 1u) uf_union(parent, (uint32_t)i, (uint32_t)right_of(x, y, L));
            if (bonds[i] & 2u) uf_union(parent, (uint32_t)i, (uint32_t)down_of(x, y, L));
        }
    }
    uint64_t n_clusters = 0;
    for (uint64_t i = 0; i < N; ++i) {
        uint32_t r = uf_find(parent, (uint32_t)i);
        label[i] = (int64_t)r;
        if (r == i) ++n_clusters;
    }
    free(parent);
    return n_clusters;
}

/* ------------------------------------------------------------------------- */
/* O6. Flip.  Coin of a cluster with canonical label rho: one Philox call    */
/* serves 128 consecutive labels: f(rho) = bit (rho mod 128) of the 128-bit    */
/* output of rng(seed, rho div 128, t, FLIP), i.e. bit (rho & 31) of word       */
/* (rho >> 5) & 3.  A flipped site is reflected across                         */
/* the line perpendicular to r:  theta -> 2 phi + pi - theta (mod 2 pi), i.e.  */
/* s -> s - 2 (s.r) r.  Specified to the rounding: only fp64 add/sub and one   */
/* fp64 -> fp32 conversion (round to nearest even).                            */
/* ------------------------------------------------------------------------- */
int xyo_flip_coin(uint64_t seed, uint64_t rho, uint64_t t)
{
    uint32_t w[4];
    xyo_rng(seed, rho >> 7, t, XYO_TAG_FLIP, w);
    return (int)((w[(rho >> 5) & 3u] >> (rho & 31u)) & 1u);
}

double xyo_reflect_const(double phi)
{
    double A = 2.0 * phi + XYO_PI;
    while (A >= XYO_TWO_PI) A -= XYO_TWO_PI;
    return A;
}

float xyo_reflect(float theta, double A)
{
    double d = A - (double)theta;
    while (d < 0.0) d += XYO_TWO_PI;
    return (float)d;
}

/* flip_site[i] != 0 -> reflect site i (injectable form).                      */
void xyo_flip_sites(float *theta, uint64_t N, double phi, const uint8_t *flip_site)
{
    double A = xyo_reflect_const(phi);
    for (uint64_t i = 0; i < N; ++i)
        if (flip_site[i]) theta[i] = xyo_reflect(theta[i], A);
}

/* the sweep's form: coin from the RNG, keyed by the canonical label.          */
uint64_t xyo_flip(float *theta, uint32_t L32, const int64_t *label, double phi,
                  uint64_t seed, uint64_t t)
{
    uint64_t N = (uint64_t)L32 * L32, n_flipped = 0;
    double A = xyo_reflect_const(phi);
    for (uint64_t i = 0; i < N; ++i) {
        if (xyo_flip_coin(seed, (uint64_t)label[i], t)) {
            theta[i] = xyo_reflect(theta[i], A);
            ++n_flipped;
        }
    }
    return n_flipped;
}

/* ------------------------------------------------------------------------- */
/* O7. Observables of a configuration (PAPER.md:40 Eq. 3; :48-54 Eq. 5-6;      */
/* :107 Eq. 9), un-normalised sums, every term in fp64, Neumaier-compensated.  */
/* ------------------------------------------------------------------------- */
typedef struct {
    uint64_t sweep;
    double   beta;
    double   E, Mx, My;
    double   Cx, Sx, Cy, Sy;
    uint64_t n_bonds_x, n_bonds_y, n_clusters;
} xyo_obs;

typedef struct { double s, c; } nsum;
static void nadd(nsum *a, double v)
{
    double t = a->s + v;
    if (fabs(a->s) >= fabs(v)) a->c += (a->s - t) + v;
    else                       a->c += (v - t) + a->s;
    a->s = t;
}
static double nval(const nsum *a) { return a->s + a->c; }

void xyo_observe(const float *theta, uint32_t L32, xyo_obs *o)
{
    uint64_t L = L32;
    nsum mx = {0, 0}, my = {0, 0}, cx = {0, 0}, sx = {0, 0}, cy = {0, 0}, sy = {0, 0};
    for (uint64_t y = 0; y < L; ++y) {
        for (uint64_t x = 0; x < L; ++x) {
            double ti = (double)theta[y * L + x];
            double tr = (double)theta[right_of(x, y, L)];
            double td = (double)theta[down_of(x, y, L)];
            nadd(&mx, cos(ti));
            nadd(&my, sin(ti));
            nadd(&cx, cos(ti - tr));
            nadd(&sx, sin(ti - tr));
            nadd(&cy, cos(ti - td));
            nadd(&sy, sin(ti - td));
        }
    }
    o->Mx = nval(&mx); o->My = nval(&my);
    o->Cx = nval(&cx); o->Sx = nval(&sx);
    o->Cy = nval(&cy); o->Sy = nval(&sy);
    o->E = -(o->Cx + o->Cy);
}

/* ------------------------------------------------------------------------- */
/* O9 (next row after the hot path: second-moment correlation length,          */
/* PAPER.md:100-107 Eq. 8-9).  Structure-factor sums at the smallest wave      */
/* vectors k = 2 pi / L along x and along y, every term in fp64:               */
/*   F[0..3] = sum_r ( cos th cos kx, cos th sin kx, sin th cos kx, sin th sin kx ) */
/*   F[4..7] = the same with ky in place of kx,   phase = 2pi64 * (x / L).     */
/* Then sum_r s(r) e^{ikr} has |.|^2 = F0^2 + F1^2 + F2^2 + F3^2 (x direction). */
/* Eq. 9 as printed squares the average; the standard estimator, used here and */
/* consistent with chi(0) = N <m^2> of Eq. 10, averages the square:            */
/*   chi(k) = < |sum_r s(r) e^{ikr}|^2 > / N   (reading G21).        */
/* ------------------------------------------------------------------------- */
void xyo_fourier(const float *theta, uint32_t L32, double F[8])
{
    uint64_t L = L32;
    nsum f[8];
    for (int k = 0; k < 8; ++k) { f[k].s = 0.0; f[k].c = 0.0; }
    for (uint64_t y = 0; y < L; ++y) {
        double ay = XYO_TWO_PI * ((double)y / (double)L);
        double cy = cos(ay), sy = sin(ay);
        for (uint64_t x = 0; x < L; ++x) {
            double ax = XYO_TWO_PI * ((double)x / (double)L);
            double cx = cos(ax), sx = sin(ax);
            double ti = (double)theta[y * L + x];
            double c = cos(ti), s = sin(ti);
            nadd(&f[0], c * cx); nadd(&f[1], c * sx); nadd(&f[2], s * cx); nadd(&f[3], s * sx);
            nadd(&f[4], c * cy); nadd(&f[5], c * sy); nadd(&f[6], s * cy); nadd(&f[7], s * sy);
        }
    }
    for (int k = 0; k < 8; ++k) F[k] = nval(&f[k]);
}

/* |sum_r s(r) e^{ikr}|^2 / N of ONE configuration from its four sums          */
double xyo_sk(const double F4[4], uint32_t L32)
{
    double N = (double)L32 * (double)L32;
    return (F4[0] * F4[0] + F4[1] * F4[1] + F4[2] * F4[2] + F4[3] * F4[3]) / N;
}

/* Eq. 8: xi_2nd(L) = sqrt(chi(0)/chi(2pi/L) - 1) / (2 sin(pi/L))              */
double xyo_xi2nd(double chi0, double chik, uint32_t L32)
{
    return sqrt(chi0 / chik - 1.0) / (2.0 * sin(XYO_PI / (double)L32));
}

/* ------------------------------------------------------------------------- */
/* One whole sweep at sweep counter t: O3 -> O4 -> O5 -> O6 -> O7.             */
/* bonds (N bytes) and label (N int64) are caller-provided scratch / outputs.  */
/* fix_phi != 0: use phi_fixed instead of the RNG direction (Ising-limit and   */
/* 2x2 tests).  Returns 0, or -1 on allocation failure.                        */
/* ------------------------------------------------------------------------- */
int xyo_sweep(float *theta, uint32_t L, uint64_t seed, uint64_t t, double beta,
              int fix_phi, double phi_fixed, uint8_t *bonds, int64_t *label, xyo_obs *o)
{
    uint64_t N = (uint64_t)L * L;
    double phi = fix_phi ? phi_fixed : xyo_phi(seed, t);
    xyo_bonds(theta, L, beta, phi, seed, t, bonds, NULL, NULL);
    uint64_t nc = xyo_label(bonds, L, label);
    if (nc == (uint64_t)-1) return -1;
    xyo_flip(theta, L, label, phi, seed, t);
    if (o) {
        uint64_t nbx = 0, nby = 0;
        for (uint64_t i = 0; i < N; ++i) { nbx += bonds[i] & 1u; nby += (bonds[i] >> 1) & 1u; }
        xyo_observe(theta, L, o);
        o->sweep = t + 1;
        o->beta = beta;
        o->n_bonds_x = nbx; o->n_bonds_y = nby; o->n_clusters = nc;
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* O8. PCC driver on the helicity modulus.             */
/* The controller is a pure state machine fed one (Cx,Sx,Cy,Sy) per sweep so   */
/* that tests can inject a synthetic observable.                               */
/* ------------------------------------------------------------------------- */
typedef struct {
    uint64_t n_sweeps, discard;
    uint32_t window, dirs;
    double   dbeta0;
    uint64_t halve_every;
    double   dbeta_min, target;
} xyo_pcc_schedule;

typedef struct {
    double   beta, dbeta;
    double   acc_e, acc_s2;
    uint64_t k;                 /* measured sweeps so far (after the discard) */
    uint64_t n_decisions;
    double   stage_sum, last_sum;       /* beta sums of the current / previous stage */
    uint64_t stage_cnt, last_cnt;
    double   last_bY;
} xyo_pcc_ctrl;

void xyo_pcc_init(xyo_pcc_ctrl *c, double beta0, double dbeta0)
{
    memset(c, 0, sizeof *c);
    c->beta = beta0;
    c->dbeta = dbeta0;
}

/* Feed the link sums of the state after one measured sweep run at c->beta.
 * Returns 1 if a decision was taken on this sweep (then *beta_dec, *bY_dec hold
 * the beta the window ran at and its beta*Upsilon estimate), else 0.
 * c->beta is the beta of the next sweep on return.                            */
int xyo_pcc_feed(xyo_pcc_ctrl *c, const xyo_pcc_schedule *s, double N,
                 double Cx, double Sx, double Cy, double Sy,
                 double *beta_dec, double *bY_dec)
{
    double e, s2;
    int decided = 0;
    if (s->dirs == 2) {
        e = (Cx + Cy) / (2.0 * N);
        double sx2 = Sx * Sx, sy2 = Sy * Sy;
        s2 = (sx2 + sy2) / ((2.0 * N) * N);
    } else {
        e = Cx / N;
        double sx = Sx / N;
        s2 = sx * sx;
    }
    c->k += 1;
    c->acc_e += e;
    c->acc_s2 += s2;
    if (c->k % s->window == 0) {
        double w = (double)s->window;
        double ae = c->acc_e / w;
        double as2 = c->acc_s2 / w;
        double bn = c->beta * N;
        double Y = ae - bn * as2;
        double bY = c->beta * Y;
        if (beta_dec) *beta_dec = c->beta;
        if (bY_dec) *bY_dec = bY;
        c->last_bY = bY;
        c->stage_sum += c->beta;
        c->stage_cnt += 1;
        c->n_decisions += 1;
        c->beta = (bY < s->target) ? c->beta + c->dbeta : c->beta - c->dbeta;
        c->acc_e = 0.0;
        c->acc_s2 = 0.0;
        decided = 1;
    }
    if (s->halve_every && c->k % s->halve_every == 0) {
        double h = c->dbeta / 2.0;
        double nd = h > s->dbeta_min ? h : s->dbeta_min;
        if (nd != c->dbeta) {
            if (c->stage_cnt > 0) { c->last_sum = c->stage_sum; c->last_cnt = c->stage_cnt; }
            c->stage_sum = 0.0;
            c->stage_cnt = 0;
        }
        c->dbeta = nd;
    }
    return decided;
}

/* mean of beta over the decisions of the last stage that has any.             */
double xyo_pcc_beta_mean(const xyo_pcc_ctrl *c)
{
    if (c->stage_cnt > 0) return c->stage_sum / (double)c->stage_cnt;
    if (c->last_cnt > 0) return c->last_sum / (double)c->last_cnt;
    return c->beta;
}

typedef struct {
    double   beta_final, dbeta_final, beta_mean;
    uint64_t n_decisions;
    double  *trace_beta, *trace_bY;
    uint64_t trace_cap, trace_len;
} xyo_pcc_out;

/* Whole PCC run on theta starting at sweep counter t0.  Returns 0 / -1.       */
int xyo_pcc_run(float *theta, uint32_t L, uint64_t seed, uint64_t t0, double beta0,
                double dbeta0, const xyo_pcc_schedule *s, xyo_pcc_out *out)
{
    uint64_t N = (uint64_t)L * L;
    uint8_t *bonds = (uint8_t *)malloc(N);
    int64_t *label = (int64_t *)malloc(N * sizeof(int64_t));
    if (!bonds || !label) { free(bonds); free(label); return -1; }
    xyo_pcc_ctrl c;
    xyo_pcc_init(&c, beta0, dbeta0);
    out->trace_len = 0;
    uint64_t t = t0;
    for (uint64_t n = 0; n < s->n_sweeps; ++n, ++t) {
        xyo_obs o;
        if (xyo_sweep(theta, L, seed, t, c.beta, 0, 0.0, bonds, label, &o)) {
            free(bonds); free(label); return -1;
        }
        if (n < s->discard) continue;
        double bdec, bY;
        if (xyo_pcc_feed(&c, s, (double)N, o.Cx, o.Sx, o.Cy, o.Sy, &bdec, &bY)) {
            if (out->trace_beta && out->trace_bY && out->trace_len < out->trace_cap) {
                out->trace_beta[out->trace_len] = bdec;
                out->trace_bY[out->trace_len] = bY;
            }
            out->trace_len += 1;
        }
    }
    out->beta_final = c.beta;
    out->dbeta_final = c.dbeta;
    out->beta_mean = xyo_pcc_beta_mean(&c);
    out->n_decisions = c.n_decisions;
    free(bonds); free(label);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Convenience for long statistical pins: n sweeps at fixed beta, returning    */
/* the per-sweep series (obs[n]).  fix_phi as in xyo_sweep.                     */
/* ------------------------------------------------------------------------- */
int xyo_run(float *theta, uint32_t L, uint64_t seed, uint64_t t0, double beta,
            uint64_t n, int fix_phi, double phi_fixed, xyo_obs *series)
{
    uint64_t N = (uint64_t)L * L;
    uint8_t *bonds = (uint8_t *)malloc(N);
    int64_t *label = (int64_t *)malloc(N * sizeof(int64_t));
    if (!bonds || !label) { free(bonds); free(label); return -1; }
    for (uint64_t k = 0; k < n; ++k) {
        if (xyo_sweep(theta, L, seed, t0 + k, beta, fix_phi, phi_fixed, bonds, label,
                      series ? &series[k] : NULL)) {
            free(bonds); free(label); return -1;
        }
    }
    free(bonds); free(label);
    return 0;
}

/* ========================================================================= */
/* q-state Potts model on the same labeling / cluster-update core             */
/* (PAPER.md:30-34 cites the authors' Potts / Ising SW     */
/* codes, refs 19 and 22, without restating the rule: the textbook            */
/* Swendsen-Wang update of PAPER.md:22's reference is used, readings P1-P5    */
/* in DESIGN.md).                                                             */
/*   H = -J sum_<ij> delta(s_i, s_j), J = 1, s_i in {0..q-1}, L x L periodic. */
/*   P1 init   cold: all 0; hot: s_i = floor(q * w0 / 2^32), w = rng(seed, i, */
/*             0, INIT).                                                      */
/*   P2 bonds  bond <ij> active iff s_i == s_j and u < p, p = 1 - exp(-beta)  */
/*             (fp64, -expm1(-beta)); u = the site's bond uniform of O1.      */
/*   P3 label  O5 (minimum site index).                                       */
/*   P4 spins  every cluster takes a fresh spin, uniform on {0..q-1}:         */
/*             s = floor(q * w / 2^32), w = word (rho & 3) of                 */
/*             rng(seed, rho >> 2, t, POTTS), rho the cluster's label.        */
/*   P5 observe E = -#{links with equal spins} (x and y links), n_k = number  */
/*             of sites with spin k.                                          */
/* ========================================================================= */
enum { XYO_TAG_POTTS = 5 };

typedef struct {
    uint64_t sweep;
    double   beta;
    int64_t  E;                 /* -(ex + ey) */
    uint64_t ex, ey;            /* links with equal spins, per direction */
    uint64_t count[16];         /* sites per spin value (q <= 16) */
    uint64_t n_bonds_x, n_bonds_y, n_clusters;
} xyo_potts_obs;

int xyo_potts_init(uint8_t *spin, uint32_t L, uint32_t q, uint64_t seed, int init)
{
    uint64_t N = (uint64_t)L * L;
    if (q < 2 || q > 16) return -1;
    if (init == 0) { memset(spin, 0, N); return 0; }
    if (init != 1) return -1;
    for (uint64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        xyo_rng(seed, i, 0, XYO_TAG_INIT, w);
        spin[i] = (uint8_t)(((uint64_t)w[0] * q) >> 32);
    }
    return 0;
}

double xyo_potts_bond_prob(double beta) { return -expm1(-beta); }

/* bonds[i]: bit0 = +x bond of site i, bit1 = +y bond */
void xyo_potts_bonds(const uint8_t *spin, uint32_t L32, double beta, uint64_t seed, uint64_t t,
                     uint8_t *bonds, uint64_t *nbx, uint64_t *nby)
{
    uint64_t L = L32, cx = 0, cy = 0;
    double p = xyo_potts_bond_prob(beta);
    for (uint64_t y = 0; y < L; ++y) {
        for (uint64_t x = 0; x < L; ++x) {
            uint64_t i = y * L + x;
            double ux, uy;
            uint8_t b = 0;
            xyo_bond_uniforms_site(seed, t, i, &ux, &uy);
            if (spin[i] == spin[right_of(x, y, L)] && ux < p) { b |= 1u; ++cx; }
            if (spin[i] == spin[down_of(x, y, L)] && uy < p) { b |= 2u; ++cy; }
            bonds[i] = b;
        }
    }
    if (nbx) *nbx = cx;
    if (nby) *nby = cy;
}

uint32_t xyo_potts_new_spin(uint64_t seed, uint64_t rho, uint64_t t, uint32_t q)
{
    uint32_t w[4];
    xyo_rng(seed, rho >> 2, t, XYO_TAG_POTTS, w);
    return (uint32_t)(((uint64_t)w[rho & 3u] * q) >> 32);
}

void xyo_potts_assign(uint8_t *spin, uint32_t L32, uint32_t q, const int64_t *label, uint64_t seed, uint64_t t)
{
    uint64_t N = (uint64_t)L32 * L32;
    for (uint64_t i = 0; i < N; ++i)
        spin[i] = (uint8_t)xyo_potts_new_spin(seed, (uint64_t)label[i], t, q);
}

void xyo_potts_observe(const uint8_t *spin, uint32_t L32, xyo_potts_obs *o)
{
    uint64_t L = L32;
    o->ex = 0; o->ey = 0;
    for (int k = 0; k < 16; ++k) o->count[k] = 0;
    for (uint64_t y = 0; y < L; ++y) {
        for (uint64_t x = 0; x < L; ++x) {
            uint64_t i = y * L + x;
            if (spin[i] == spin[right_of(x, y, L)]) ++o->ex;
            if (spin[i] == spin[down_of(x, y, L)]) ++o->ey;
            ++o->count[spin[i] & 15u];
        }
    }
    o->E = -(int64_t)(o->ex + o->ey);
}

/* one sweep at counter t; bonds / label: caller-provided scratch of N entries; obs describes the */
/* state AFTER the sweep, with the bond and cluster counts of this sweep                          */
int xyo_potts_sweep(uint8_t *spin, uint32_t L, uint32_t q, uint64_t seed, uint64_t t, double beta,
                    uint8_t *bonds, int64_t *label, xyo_potts_obs *obs)
{
    uint64_t nbx, nby, ncl;
    if (q < 2 || q > 16) return -1;
    xyo_potts_bonds(spin, L, beta, seed, t, bonds, &nbx, &nby);
    ncl = xyo_label(bonds, L, label);
    if (ncl == (uint64_t)-1) return -1;
    xyo_potts_assign(spin, L, q, label, seed, t);
    if (obs) {
        xyo_potts_observe(spin, L, obs);
        obs->sweep = t + 1; obs->beta = beta;
        obs->n_bonds_x = nbx; obs->n_bonds_y = nby; obs->n_clusters = ncl;
    }
    return 0;
}
