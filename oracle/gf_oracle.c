/*
 * gf_oracle.c -- CPU ORACLE for the SU(3) gauge-fixing relaxation sweep.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the
 * __graft_entry__.smoke() check and bench.py's cpu_baseline / --impl reference
 * legs may call it.  It shares no code, header, table or constant with the CUDA
 * path under paper_1305_3440_b200/csrc/ and neither includes the other.
 *
 * It is a plain, slow, double-precision restatement of
 *   Schroeck & Vogt, "Gauge fixing in lattice QCD with multi-GPUs"
 *   (arXiv:1305.3440; /root/reference/PAPER.md), cited below as PAPER.md:<line>.
 * The method is an iteration (a local optimisation with several valid
 * outcomes), so the oracle follows the algorithm step by step in the paper's
 * order and notation; no blocking, fusion or reordering.  Where PAPER.md is
 * silent the reading taken is listed in DESIGN.md ("Readings", A1..A20) and
 * named here next to the line that implements it.
 *
 * Conventions
 *   dims[4] = {N_t, N_x, N_y, N_z};  mu = 0 is time (PAPER.md:111 writes the
 *   temporal link U_0), mu = 1,2,3 = x,y,z.  Site s = x + N_x (y + N_y (z + N_z t)).
 *   U is the canonical array  U[s][mu][a][b]  of C99 double complex, row major,
 *   i.e. a numpy complex128 array of shape (Nt,Nz,Ny,Nx,4,3,3).
 *   parity(s) = (t + x + y + z) mod 2.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): see the list in
 * DESIGN.md section "Oracle pins"; tests/test_oracle_mutants.py re-runs them on
 * single-line mutants of this file (each must fail a pin).  Unpinned CHOICES OF
 * READING (several readings are equally valid and the paper does not decide):
 * the overall normalisation of A_mu (A1), per-SU(2)-factor overrelaxation (A7),
 * one random draw per (site, subgroup) (A8).  For those the header says: parity
 * unpinned -- the paper cannot tell the readings apart; what this file computes
 * UNDER each reading is pinned (closed forms per subgroup, the ordered product
 * of the three factors with distinct draws, every function incl. the
 * unitarity checker against fields with a known defect).
 *
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fcx-limited-range [-fopenmp]
 *        -shared -fPIC gf_oracle.c -o libgf_oracle.so -lm   (oracle/build.py)
 */
#include <complex.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cd;

enum { ORACLE_LANDAU = 0, ORACLE_COULOMB = 1 };
enum { ORACLE_RELAX = 0, ORACLE_OVERRELAX = 1, ORACLE_STOCHASTIC = 2 };

#define NC 3 /* number of colours */

/* ------------------------------------------------------------------ threads */

static int g_threads = 1;

/* Number of OpenMP threads the site loops use (1 = serial).  Returns the value
 * actually in effect (1 when built without OpenMP). */
int oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n < 1) n = omp_get_num_procs();
    g_threads = n;
#else
    (void)n;
    g_threads = 1;
#endif
    return g_threads;
}

int oracle_get_threads(void) { return g_threads; }

/* ----------------------------------------------------------------- geometry */

static size_t volume(const int dims[4])
{
    return (size_t)dims[0] * dims[1] * dims[2] * dims[3];
}

/* s -> c[mu] with c[0]=t, c[1]=x, c[2]=y, c[3]=z */
static void site_coords(const int dims[4], size_t s, int c[4])
{
    c[1] = (int)(s % dims[1]); s /= dims[1];
    c[2] = (int)(s % dims[2]); s /= dims[2];
    c[3] = (int)(s % dims[3]); s /= dims[3];
    c[0] = (int)s;
}

static size_t site_index(const int dims[4], const int c[4])
{
    return (size_t)c[1] + (size_t)dims[1] * (c[2] + (size_t)dims[2] * (c[3] + (size_t)dims[3] * c[0]));
}

/* index of x + dir*mu_hat with periodic wrap, dir = +1 or -1 */
static size_t neighbour(const int dims[4], const int c[4], int mu, int dir)
{
    int n[4] = { c[0], c[1], c[2], c[3] };
    n[mu] = (c[mu] + dir + dims[mu]) % dims[mu];
    return site_index(dims, n);
}

static int site_parity(const int c[4]) { return (c[0] + c[1] + c[2] + c[3]) & 1; }

static cd *link_ptr(cd *U, size_t s, int mu) { return U + (s * 4 + (size_t)mu) * 9; }
static const cd *link_cptr(const cd *U, size_t s, int mu) { return U + (s * 4 + (size_t)mu) * 9; }

/* first direction that enters K, F and theta: Landau sums mu = 0..3
 * (PAPER.md:39, :50, :69), Coulomb only the spatial mu = 1..3 (reading A17) */
static int first_dir(int gauge) { return gauge == ORACLE_COULOMB ? 1 : 0; }

/* ------------------------------------------------------- 3x3 complex algebra */

static void mat_mul(const cd A[9], const cd B[9], cd C[9]) /* C = A B */
{
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            cd s = 0;
            for (int k = 0; k < 3; ++k) s += A[3 * a + k] * B[3 * k + b];
            C[3 * a + b] = s;
        }
}

static void mat_dagger(const cd A[9], cd C[9]) /* C = A^dagger */
{
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) C[3 * a + b] = conj(A[3 * b + a]);
}

static void mat_identity(cd A[9])
{
    for (int k = 0; k < 9; ++k) A[k] = 0;
    A[0] = A[4] = A[8] = 1;
}

/* ------------------------------------------------ O4: Philox4x32-10 (public) */

/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3"
 * (SC'11).  The RNG is not specified by PAPER.md:84; BASELINE.json's north_star
 * asks for counter-based Philox keyed by (seed, sweep, site).  Pinned by the
 * algorithm's published known-answer vectors (tests/golden/philox4x32_10_kat.txt). */
void oracle_philox4x32_10(const uint32_t counter[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = counter[0], c1 = counter[1], c2 = counter[2], c3 = counter[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* The three uniform draws u_k in [0,1) of one site visit (reading A8: one
 * independent draw per (site, subgroup)): counter = (s_lo, s_hi,
 * half_sweep_counter, 0), key = (seed_lo, seed_hi), u_k = (word_k >> 8) * 2^-24. */
void oracle_site_uniforms(uint64_t seed, uint32_t half_sweep_counter, uint64_t s, double u[3])
{
    uint32_t ctr[4] = { (uint32_t)s, (uint32_t)(s >> 32), half_sweep_counter, 0u };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    oracle_philox4x32_10(ctr, key, w);
    for (int k = 0; k < 3; ++k) u[k] = (double)(w[k] >> 8) * (1.0 / 16777216.0);
}

/* ------------------------------------------------------- O1: functional F */

/* PAPER.md:39 (eq. 2): F = 1/(N_c N_d V) Re sum_{mu,x} tr U_mu(x), N_d = 4.
 * Landau: out[0] = F.  Coulomb (reading A2/A17): for every time slice t,
 * out[t] = 1/(N_c 3 N_s^3) Re sum_{x in slice t} sum_{mu=1..3} tr U_mu(x). */
void oracle_functional(const cd *U, const int dims[4], int gauge, double *out)
{
    const size_t V = volume(dims);
    const size_t Vs = (size_t)dims[1] * dims[2] * dims[3];
    const int mu0 = first_dir(gauge);
    const int nslice = gauge == ORACLE_COULOMB ? dims[0] : 1;
    const size_t per = gauge == ORACLE_COULOMB ? Vs : V;
    for (int t = 0; t < nslice; ++t) {
        double sum = 0.0;
        for (size_t s = t * per; s < (t + 1) * per; ++s)
            for (int mu = mu0; mu < 4; ++mu) {
                const cd *u = link_cptr(U, s, mu);
                sum += creal(u[0] + u[4] + u[8]);
            }
        out[t] = sum / ((double)NC * (4 - mu0) * (double)per);
    }
}

/* ------------------------------------------------------ O2: precision theta */

/* Reading A1 (PAPER.md:48-50 never expresses A_mu through U_mu):
 * A_mu(x) = [(U - U^dagger)/(2i)] - (1/3) tr[(U - U^dagger)/(2i)] 1. */
static void gauge_field_A(const cd u[9], cd A[9])
{
    cd ud[9];
    mat_dagger(u, ud);
    for (int k = 0; k < 9; ++k) A[k] = (u[k] - ud[k]) / (2.0 * I);
    cd tr = (A[0] + A[4] + A[8]) / 3.0;
    A[0] -= tr; A[4] -= tr; A[8] -= tr;
}

/* PAPER.md:50 (eq. 4): Delta(x) = sum_mu (A_mu(x) - A_mu(x - mu_hat)). */
void oracle_site_delta(const cd *U, const int dims[4], int gauge, size_t s, cd Delta[9])
{
    int c[4];
    site_coords(dims, s, c);
    for (int k = 0; k < 9; ++k) Delta[k] = 0;
    for (int mu = first_dir(gauge); mu < 4; ++mu) {
        cd Af[9], Ab[9];
        gauge_field_A(link_cptr(U, s, mu), Af);
        gauge_field_A(link_cptr(U, neighbour(dims, c, mu, -1), mu), Ab);
        for (int k = 0; k < 9; ++k) Delta[k] += Af[k] - Ab[k];
    }
}

/* PAPER.md:52 (eq. 5): theta = 1/(N_c V) sum_x tr[Delta(x) Delta(x)^dagger].
 * Landau: out[0].  Coulomb (A17): out[t] = 1/(N_c N_s^3) sum_{x in slice t}. */
void oracle_theta(const cd *U, const int dims[4], int gauge, double *out)
{
    const size_t V = volume(dims);
    const size_t Vs = (size_t)dims[1] * dims[2] * dims[3];
    const int nslice = gauge == ORACLE_COULOMB ? dims[0] : 1;
    const size_t per = gauge == ORACLE_COULOMB ? Vs : V;
    for (int t = 0; t < nslice; ++t) {
        double sum = 0.0;
#ifdef _OPENMP
#pragma omp parallel for reduction(+ : sum) num_threads(g_threads) schedule(static)
#endif
        for (size_t s = t * per; s < (t + 1) * per; ++s) {
            cd D[9], Dd[9], P[9];
            oracle_site_delta(U, dims, gauge, s, D);
            mat_dagger(D, Dd);
            mat_mul(D, Dd, P);
            sum += creal(P[0] + P[4] + P[8]);
        }
        out[t] = sum / ((double)NC * (double)per);
    }
}

/* ------------------------------------------------------------ O3: the sweep */

/* PAPER.md:69 (eq. 8) with the neighbours' g = 1 (reading A3: inside a sweep a
 * transformation is applied to the links at once, so the neighbours carry no
 * pending g):  K(x) = sum_mu ( U_mu(x) + U_mu(x - mu_hat)^dagger ). */
static void build_K(cd *const fwd[4], cd *const bwd[4], int gauge, cd K[9])
{
    for (int k = 0; k < 9; ++k) K[k] = 0;
    for (int mu = first_dir(gauge); mu < 4; ++mu) {
        cd bd[9];
        mat_dagger(bwd[mu], bd);
        for (int k = 0; k < 9; ++k) K[k] += fwd[mu][k] + bd[k];
    }
}

void oracle_site_K(const cd *U, const int dims[4], int gauge, size_t s, cd K[9])
{
    int c[4];
    site_coords(dims, s, c);
    cd *fwd[4], *bwd[4];
    for (int mu = 0; mu < 4; ++mu) {
        fwd[mu] = (cd *)link_cptr(U, s, mu);
        bwd[mu] = (cd *)link_cptr(U, neighbour(dims, c, mu, -1), mu);
    }
    build_K(fwd, bwd, gauge, K);
}

/* Reading A4.  PAPER.md:73 (eq. 9), g = K^dagger / sqrt(det K^dagger), is
 * stated for SU(2), where K is a real multiple of an SU(2) matrix.  The 2x2
 * block (i,j) of an SU(3) K is not; its part that matters for Re tr[a K_sub]
 * with a in SU(2) is the projection on SU(2) x R+.  Writing
 *   a = [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]]
 * one finds Re tr[a K_sub] = a . v with the 4-vector v below, i.e. the
 * projected block is P = (|v|/2) W with W in SU(2) and eq. 9 applied to P gives
 * g = P^dagger / sqrt(det P^dagger) = W^dagger, whose 4-vector is v/|v|. */
void oracle_su2_vector(const cd K[9], int i, int j, double v[4])
{
    const cd Kii = K[3 * i + i], Kij = K[3 * i + j], Kji = K[3 * j + i], Kjj = K[3 * j + j];
    v[0] = creal(Kii + Kjj);
    v[1] = -cimag(Kij + Kji);
    v[2] = creal(Kji - Kij);
    v[3] = cimag(Kjj - Kii);
}

/* From v to the SU(2) update a (unit 4-vector).
 *   RELAX       a = v/|v|                                   PAPER.md:73 (eq. 9)
 *   OVERRELAX   g^omega "to first order", reading A7: per SU(2)
 *               factor, a^omega ~ 1 + omega (a - 1), re-normalised; written
 *               with w = |v| (1 + omega (a - 1)) to avoid one division.
 *   STOCHASTIC  g -> g^2 with probability p; u is the uniform
 *               draw for this (site, subgroup) (reading A8).
 * Reading A9: |v| = 0 -> a = 1. */
void oracle_su2_update(const double v[4], int algo, double omega, double p, double u, double a[4])
{
    const double n = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + v[3] * v[3]);
    if (n == 0.0) {
        a[0] = 1.0; a[1] = a[2] = a[3] = 0.0;
        return;
    }
    if (algo == ORACLE_OVERRELAX) {
        double w[4] = { omega * v[0] + (1.0 - omega) * n, omega * v[1], omega * v[2], omega * v[3] };
        const double nw = sqrt(w[0] * w[0] + w[1] * w[1] + w[2] * w[2] + w[3] * w[3]);
        for (int k = 0; k < 4; ++k) a[k] = w[k] / nw;
        return;
    }
    for (int k = 0; k < 4; ++k) a[k] = v[k] / n;
    if (algo == ORACLE_STOCHASTIC && u < p) {
        const double a0 = a[0];
        a[0] = 2.0 * a0 * a0 - 1.0;
        a[1] = 2.0 * a0 * a[1];
        a[2] = 2.0 * a0 * a[2];
        a[3] = 2.0 * a0 * a[3];
    }
}

/* M <- E M with E the 3x3 embedding of a in the (i,j) subgroup: E = 1 except
 * E_ii = a0 + i a3, E_ij = a2 + i a1, E_ji = -a2 + i a1, E_jj = a0 - i a3. */
static void embed_left_multiply(cd M[9], int i, int j, const double a[4])
{
    const cd Eii = a[0] + I * a[3], Eij = a[2] + I * a[1];
    const cd Eji = -a[2] + I * a[1], Ejj = a[0] - I * a[3];
    for (int b = 0; b < 3; ++b) {
        const cd mi = M[3 * i + b], mj = M[3 * j + b];
        M[3 * i + b] = Eii * mi + Eij * mj;
        M[3 * j + b] = Eji * mi + Ejj * mj;
    }
}

/* "for SU(3) one iteratively operates in the three SU(2)
 * subgroups [4]".  Reading A5: order (0,1), (0,2), (1,2), one pass.  Reading
 * A6: K is refreshed between subgroups (K <- E K), g accumulates (g <- E g). */
void oracle_site_g(const cd K_in[9], int algo, double omega, double p, const double u[3], cd g[9])
{
    static const int sub[3][2] = { { 0, 1 }, { 0, 2 }, { 1, 2 } };
    cd K[9];
    for (int k = 0; k < 9; ++k) K[k] = K_in[k];
    mat_identity(g);
    for (int k = 0; k < 3; ++k) {
        double v[4], a[4];
        oracle_su2_vector(K, sub[k][0], sub[k][1], v);
        oracle_su2_update(v, algo, omega, p, u[k], a);
        embed_left_multiply(K, sub[k][0], sub[k][1], a);
        embed_left_multiply(g, sub[k][0], sub[k][1], a);
    }
}

/* One site visit: K (eq. 8), g (eq. 9 per subgroup), then PAPER.md:43 (eq. 3)
 * with g = 1 on the other parity:  U_mu(x) <- g U_mu(x),
 * U_mu(x - mu_hat) <- U_mu(x - mu_hat) g^dagger, for all four mu -- also in
 * Coulomb gauge (A17), else it would not be a gauge transformation. */
static void update_site(cd *const fwd[4], cd *const bwd[4], int gauge, int algo,
                        double omega, double p, const double u[3], cd g_out[9])
{
    cd K[9], g[9], gd[9], tmp[9];
    build_K(fwd, bwd, gauge, K);
    oracle_site_g(K, algo, omega, p, u, g);
    mat_dagger(g, gd);
    for (int mu = 0; mu < 4; ++mu) {
        mat_mul(g, fwd[mu], tmp);
        for (int k = 0; k < 9; ++k) fwd[mu][k] = tmp[k];
        mat_mul(bwd[mu], gd, tmp);
        for (int k = 0; k < 9; ++k) bwd[mu][k] = tmp[k];
    }
    if (g_out)
        for (int k = 0; k < 9; ++k) g_out[k] = g[k];
}

/* The same site visit on a free-standing bundle of the 8 links that touch one
 * site (fwd[mu] = U_mu(x), bwd[mu] = U_mu(x - mu_hat)); used to check sampled
 * sites of lattices too large to sweep on the host. */
void oracle_update_links8(cd fwd[4][9], cd bwd[4][9], int gauge, int algo,
                          double omega, double p, const double u[3], cd g_out[9])
{
    cd *f[4] = { fwd[0], fwd[1], fwd[2], fwd[3] };
    cd *b[4] = { bwd[0], bwd[1], bwd[2], bwd[3] };
    update_site(f, b, gauge, algo, omega, p, u, g_out);
}

/* Gtot (may be NULL): the accumulated transformation, one 3x3 matrix per site,
 * Gtot[s][a][b].  A site visit applies g(x) on top of what was applied before,
 * so by PAPER.md:43 (eq. 3) the total transformation becomes g(x) Gtot(x). */
static void visit_site(cd *U, cd *Gtot, const int *slice_active, const int dims[4], int gauge, int parity, int algo,
                       double omega, double p, uint64_t seed, uint32_t half_sweep_counter, size_t s)
{
    int c[4];
    site_coords(dims, s, c);
    if (site_parity(c) != parity) return;
    if (slice_active && !slice_active[c[0]]) return;   /* frozen time slice (Coulomb, reading A17b) */
    cd *fwd[4], *bwd[4];
    for (int mu = 0; mu < 4; ++mu) {
        fwd[mu] = link_ptr(U, s, mu);
        bwd[mu] = link_ptr(U, neighbour(dims, c, mu, -1), mu);
    }
    double u[3] = { 0.0, 0.0, 0.0 };
    if (algo == ORACLE_STOCHASTIC) oracle_site_uniforms(seed, half_sweep_counter, (uint64_t)s, u);
    cd g[9], tmp[9];
    update_site(fwd, bwd, gauge, algo, omega, p, u, g);
    if (Gtot) {
        mat_mul(g, Gtot + s * 9, tmp);
        for (int k = 0; k < 9; ++k) Gtot[s * 9 + k] = tmp[k];
    }
}

/* all sites of one parity subset can be optimised at the same
 * time; the sites are visited in lexicographic order (reverse_order != 0: in
 * the opposite order -- same-parity sites share no link, so the result must be
 * bitwise the same; that is one of the pins). */
static void sweep_impl(cd *U, cd *Gtot, const int *slice_active, const int dims[4], int gauge, int parity, int algo, double omega,
                       double p, uint64_t seed, uint32_t half_sweep_counter, int reverse_order)
{
    const size_t V = volume(dims);
    if (reverse_order) {
        for (size_t k = V; k-- > 0;)
            visit_site(U, Gtot, slice_active, dims, gauge, parity, algo, omega, p, seed, half_sweep_counter, k);
        return;
    }
#ifdef _OPENMP
#pragma omp parallel for num_threads(g_threads) schedule(static)
#endif
    for (size_t s = 0; s < V; ++s)
        visit_site(U, Gtot, slice_active, dims, gauge, parity, algo, omega, p, seed, half_sweep_counter, s);
}

void oracle_sweep_ordered(cd *U, const int dims[4], int gauge, int parity, int algo, double omega,
                          double p, uint64_t seed, uint32_t half_sweep_counter, int reverse_order)
{
    sweep_impl(U, NULL, NULL, dims, gauge, parity, algo, omega, p, seed, half_sweep_counter, reverse_order);
}

/* The same half-sweep, also recording the transformation: Gtot(x) <- g(x) Gtot(x)
 * on the visited sites.  Starting from Gtot = 1 the swept links always equal
 * Gtot(x) U^(0)_mu(x) Gtot(x + mu_hat)^dagger of the initial links U^(0) (eq. 3);
 * that identity is one of the pins. */
void oracle_sweep_accumulate(cd *U, cd *Gtot, const int dims[4], int gauge, int parity, int algo,
                             double omega, double p, uint64_t seed, uint32_t half_sweep_counter)
{
    sweep_impl(U, Gtot, NULL, dims, gauge, parity, algo, omega, p, seed, half_sweep_counter, 0);
}

/* Reading A17b (an option beside A17; PAPER.md:11, :29 only name Coulomb gauge): time slices
 * are fixed independently -- in Coulomb gauge K, F_t and theta_t of slice t involve only the
 * spatial links of slice t, which only the sites of slice t change -- so a slice whose theta_t
 * has reached the target may stop being swept ("frozen").  slice_active[t] != 0: the sites of
 * slice t are visited; 0: skipped.  Gtot may be NULL. */
void oracle_sweep_masked(cd *U, cd *Gtot, const int *slice_active, const int dims[4], int gauge, int parity,
                         int algo, double omega, double p, uint64_t seed, uint32_t half_sweep_counter)
{
    sweep_impl(U, Gtot, slice_active, dims, gauge, parity, algo, omega, p, seed, half_sweep_counter, 0);
}

/* PAPER.md:43 (eq. 3) written out: U_out_mu(x) = G(x) U_mu(x) G(x + mu_hat)^dagger. */
void oracle_apply_transform(const cd *U, const cd *G, const int dims[4], cd *U_out)
{
    const size_t V = volume(dims);
    for (size_t s = 0; s < V; ++s) {
        int c[4];
        site_coords(dims, s, c);
        for (int mu = 0; mu < 4; ++mu) {
            cd gd[9], tmp[9];
            mat_dagger(G + neighbour(dims, c, mu, +1) * 9, gd);
            mat_mul(G + s * 9, link_cptr(U, s, mu), tmp);
            mat_mul(tmp, gd, U_out + (s * 4 + (size_t)mu) * 9);
        }
    }
}

void oracle_sweep(cd *U, const int dims[4], int gauge, int parity, int algo, double omega,
                  double p, uint64_t seed, uint32_t half_sweep_counter)
{
    oracle_sweep_ordered(U, dims, gauge, parity, algo, omega, p, seed, half_sweep_counter, 0);
}

/* --------------------------------------------------------- O5: the fix loop */

/* "The two parity sublattices are treated consecutively and the
 * relaxation algorithm is iterated until the requested gauge precision theta
 * has been reached."  Readings A10/A11: iteration it = 1,2,.. is parity 0 then
 * parity 1 with half-sweep counters first_counter + 2(it-1), +1; theta is
 * evaluated after iterations that are multiples of check_every and after the
 * last one; Coulomb stops when max_t theta_t < target.  Returns the number of
 * iterations done; *theta_out = theta (Coulomb: max_t theta_t) at the last
 * evaluation; *converged = 1 if it fell below the target. */
int oracle_fix_until(cd *U, const int dims[4], int gauge, int algo, double omega, double p,
                     uint64_t seed, uint32_t first_counter, double theta_target, int max_iter,
                     int check_every, double *theta_out, int *converged)
{
    double th[4096];
    const int nslice = gauge == ORACLE_COULOMB ? dims[0] : 1;
    double theta = INFINITY;
    *converged = 0;
    *theta_out = INFINITY;
    if (nslice > 4096) return -1;              /* th[] holds one theta_t per time slice: refuse, do not overrun */
    int it = 0;
    if (check_every < 1) check_every = 1;
    while (it < max_iter) {
        oracle_sweep(U, dims, gauge, 0, algo, omega, p, seed, first_counter + 2u * (uint32_t)it);
        oracle_sweep(U, dims, gauge, 1, algo, omega, p, seed, first_counter + 2u * (uint32_t)it + 1u);
        ++it;
        if (it % check_every == 0 || it == max_iter) {
            oracle_theta(U, dims, gauge, th);
            theta = th[0];
            for (int t = 1; t < nslice && t < 4096; ++t)
                if (th[t] > theta) theta = th[t];
            if (theta < theta_target) { *converged = 1; break; }
        }
    }
    *theta_out = theta;
    return it;
}

/* The fix loop of oracle_fix_until for Coulomb gauge with slice freezing (A17b): after every
 * theta evaluation the slices with theta_t < target are frozen for the rest of the run; the
 * run ends when all are frozen.  theta_slices[t] = theta_t at the last evaluation (a frozen
 * slice keeps its value: nothing that enters it changes any more); frozen_at[t] = iteration at
 * which slice t was frozen (0 = never).  Returns the iterations done. */
int oracle_fix_until_freeze(cd *U, const int dims[4], int algo, double omega, double p, uint64_t seed,
                            uint32_t first_counter, double theta_target, int max_iter, int check_every,
                            double *theta_slices, int *frozen_at, int *converged)
{
    int active[4096];
    const int nt = dims[0];
    *converged = 0;
    if (nt > 4096) return -1;                  /* active[] holds one flag per time slice: refuse, do not overrun */
    for (int t = 0; t < nt; ++t) { active[t] = 1; frozen_at[t] = 0; }
    int it = 0;
    if (check_every < 1) check_every = 1;
    while (it < max_iter) {
        oracle_sweep_masked(U, NULL, active, dims, ORACLE_COULOMB, 0, algo, omega, p, seed, first_counter + 2u * (uint32_t)it);
        oracle_sweep_masked(U, NULL, active, dims, ORACLE_COULOMB, 1, algo, omega, p, seed, first_counter + 2u * (uint32_t)it + 1u);
        ++it;
        if (it % check_every == 0 || it == max_iter) {
            oracle_theta(U, dims, ORACLE_COULOMB, theta_slices);
            int left = 0;
            for (int t = 0; t < nt; ++t) {
                if (active[t] && theta_slices[t] < theta_target) { active[t] = 0; frozen_at[t] = it; }
                left += active[t];
            }
            if (left == 0) { *converged = 1; break; }
        }
    }
    return it;
}

/* ------------------------------------------------------------ O6: diagnostics */

/* Mean plaquette, gauge invariant:
 * P = 1/(6 N_c V) sum_x sum_{mu<nu} Re tr[U_mu(x) U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger]. */
double oracle_plaquette(const cd *U, const int dims[4])
{
    const size_t V = volume(dims);
    double sum = 0.0;
#ifdef _OPENMP
#pragma omp parallel for reduction(+ : sum) num_threads(g_threads) schedule(static)
#endif
    for (size_t s = 0; s < V; ++s) {
        int c[4];
        site_coords(dims, s, c);
        for (int mu = 0; mu < 4; ++mu)
            for (int nu = mu + 1; nu < 4; ++nu) {
                cd t1[9], t2[9], d1[9], d2[9], P[9];
                mat_mul(link_cptr(U, s, mu), link_cptr(U, neighbour(dims, c, mu, +1), nu), t1);
                mat_dagger(link_cptr(U, neighbour(dims, c, nu, +1), mu), d1);
                mat_dagger(link_cptr(U, s, nu), d2);
                mat_mul(t1, d1, t2);
                mat_mul(t2, d2, P);
                sum += creal(P[0] + P[4] + P[8]);
            }
    }
    return sum / (6.0 * NC * (double)V);
}

/* out[0] = max over links and entries of |U U^dagger - 1|, out[1] = max |det U - 1|. */
void oracle_unitarity_defect(const cd *U, const int dims[4], double out[2])
{
    const size_t nlinks = volume(dims) * 4;
    double dmax = 0.0, detmax = 0.0;
    for (size_t l = 0; l < nlinks; ++l) {
        const cd *u = U + l * 9;
        cd ud[9], P[9];
        mat_dagger(u, ud);
        mat_mul(u, ud, P);
        P[0] -= 1; P[4] -= 1; P[8] -= 1;
        for (int k = 0; k < 9; ++k)
            if (cabs(P[k]) > dmax) dmax = cabs(P[k]);
        cd det = u[0] * (u[4] * u[8] - u[5] * u[7]) - u[1] * (u[3] * u[8] - u[5] * u[6])
               + u[2] * (u[3] * u[7] - u[4] * u[6]);
        if (cabs(det - 1) > detmax) detmax = cabs(det - 1);
    }
    out[0] = dmax;
    out[1] = detmax;
}
