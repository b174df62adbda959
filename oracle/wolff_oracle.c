/*
 * wolff_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, sequential CPU statement of what the hot path of
 * Komura & Okabe, "GPU-based single-cluster algorithm for the simulation of
 * the Ising model" (arXiv 1110.0899; /root/reference/PAPER.md) computes:
 * one Wolff single-cluster update on a periodic 2D square / 3D simple-cubic
 * Ising lattice, repeated.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call into this file.
 * It shares no code, header, table or constant generator with the CUDA path
 * under paper_1110_0899_b200/csrc/ and neither includes the other.
 *
 * Paper passages followed (PAPER.md line numbers):
 *   Hamiltonian, periodic boundaries ............ :36-40  (section 2, Eq. 2)
 *   steps (i)-(v) of the single-cluster update .. :42-48  (section 2)
 *   termination "in < ic" / flip-timing freedom . :50     (section 2)
 *   add probability p = 1 - exp(-2 beta) ........ :120    (section 4; the
 *        minus sign is lost at :45-46, reading G1/R1 in DESIGN.md)
 *   E and M "measurement" ....................... :126    (section 5)
 *
 * Where the paper is silent the readings R1..R15 of DESIGN.md section 3 are
 * taken; each is restated next to the function that implements it.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   philox4x32_10 ........ published known-answer vectors (tests/golden/)
 *   threshold ............ exact integer closed form at 2D T_c, limits
 *   site draw ............ range, power-of-two exactness, chi^2
 *   nbr / edge ownership . brute-force involution + double cover
 *   run (cluster) ........ independent union-find over all bonds; p=0, p=1
 *                          flood fill; invariants
 *   run (sampler) ........ exact enumeration of 4x4 (2^16) and 3x3x3 (2^27)
 *                          within 3 standard errors; <|C|> = <M^2>/N;
 *                          Kaufman's exact finite-torus energy; Onsager band
 *   observables .......... closed forms (cold lattice, checkerboard, stripes)
 *   moments / binder ..... hand-computed series, Python big integers past 2^64,
 *                          |M| = N gives U = 2/3, Gaussian M gives U -> 0, exact
 *                          4x4 / 3x3x3 enumeration (U = 0.61719932 at 2D T_c)
 * No function in this file is "parity unpinned".
 *
 * Precision: everything is integer except the threshold, which is IEEE
 * double as fixed in reading R7.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- Philox */

/* Philox4x32-10 of Salmon, Moraes, Dror, Shaw (SC'11), reading R11:
 * round:  (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
 * with M0 = 0xD2511F53, M1 = 0xCD9E8D57; between rounds the key is bumped by
 * (0x9E3779B9, 0xBB67AE85); ten rounds, nine bumps. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) {
            k0 += 0x9E3779B9u;
            k1 += 0xBB67AE85u;
        }
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(prod1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)prod1;
        uint32_t n2 = (uint32_t)(prod0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)prod0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Domain tags in bits 31:30 of counter word 1 keep the three streams the
 * method draws from disjoint (reading R10). */
#define DOMAIN_BOND 0u
#define DOMAIN_SITE 1u
#define DOMAIN_INIT 2u

/* ------------------------------------------------------------- threshold */

/* Reading R7 (p = 1 - e^{-2 beta}, beta = J/T): p in IEEE
 * double as -expm1(-2J/T); thr = floor(p * 2^32) in [0, 2^32]; a bond is
 * active iff its 32-bit Philox word, widened to 64 bits, is < thr. */
uint64_t oracle_threshold(double J, double T)
{
    double p = -expm1(-2.0 * J / T);
    if (p <= 0.0) return 0;
    double scaled = floor(p * 4294967296.0);
    if (scaled >= 4294967296.0) return 4294967296ull;
    return (uint64_t)scaled;
}

/* ------------------------------------------------------ lattice indexing */

/* Reading R5: site id i = x + L*y (+ L*L*z), x fastest; direction d = 0,1,2
 * is x,y,z; the neighbour in direction (d, sign) has coordinate d replaced
 * by (c_d +/- 1) mod L  (periodic boundaries). */
uint64_t oracle_nbr(int dim, int L, uint64_t i, int d, int sign)
{
    uint64_t c[3];
    uint64_t rest = i;
    for (int k = 0; k < dim; ++k) {
        c[k] = rest % (uint64_t)L;
        rest /= (uint64_t)L;
    }
    if (sign > 0) c[d] = (c[d] + 1) % (uint64_t)L;
    else          c[d] = (c[d] + (uint64_t)L - 1) % (uint64_t)L;
    uint64_t j = 0;
    for (int k = dim - 1; k >= 0; --k) j = j * (uint64_t)L + c[k];
    return j;
}

/* ------------------------------------------------------- random decisions */

/* Reading R8 ("Choose a site i randomly"): uniform on [0, N):
 * x = Philox(key = seed, ctr = (0, SITE<<30, u_lo, u_hi)); r = x0 | x1<<32;
 * i0 = floor(r * N / 2^64). */
uint64_t oracle_site_draw(uint64_t seed, uint64_t u, uint64_t N)
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { 0u, DOMAIN_SITE << 30, (uint32_t)u, (uint32_t)(u >> 32) };
    uint32_t x[4];
    oracle_philox4x32_10(ctr, key, x);
    uint64_t r = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
    return (uint64_t)(((unsigned __int128)r * (unsigned __int128)N) >> 64);
}

/* Readings R6 + R10: the undirected bond between `owner` and its neighbour in
 * direction +d is edge (owner, d).  Its bond variable for update u is word d
 * of Philox(key = seed, ctr = (owner_lo, BOND<<30 | owner_hi, u_lo, u_hi));
 * the bond is active iff that word < thr.  A function of (seed, u, edge)
 * only, so traversal order cannot show (PAPER.md:50 notes this freedom). */
int oracle_bond_active(uint64_t seed, uint64_t u, uint64_t owner, int d, uint64_t thr)
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)owner, (DOMAIN_BOND << 30) | (uint32_t)(owner >> 32),
                        (uint32_t)u, (uint32_t)(u >> 32) };
    uint32_t x[4];
    oracle_philox4x32_10(ctr, key, x);
    return (uint64_t)x[d] < thr;
}

/* Reading R9 ("random +/-1 start from seed", BASELINE.json configs): site i
 * takes bit (i mod 128) of Philox(key = seed, ctr = (b_lo, INIT<<30 | b_hi,
 * 0, 0)) with b = i div 128; the bit is bit (i mod 32) of word ((i div 32)
 * mod 4); 1 -> +1, 0 -> -1. */
int oracle_init_spin(uint64_t seed, uint64_t i)
{
    uint64_t b = i >> 7;
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)b, (DOMAIN_INIT << 30) | (uint32_t)(b >> 32), 0u, 0u };
    uint32_t x[4];
    oracle_philox4x32_10(ctr, key, x);
    uint32_t word = x[(i >> 5) & 3u];
    return ((word >> (i & 31u)) & 1u) ? +1 : -1;
}

/* ------------------------------------------------------------------ state */

typedef struct oracle_ctx {
    int dim, L;
    uint64_t N;
    double J, T;
    uint64_t seed;
    uint64_t thr;
    uint64_t u;        /* global update index, reading R12: never reset */
    int8_t *s;         /* N spins, +1 / -1 */
    uint64_t *stack;   /* a site is pushed at most once per update */
} oracle_ctx;

oracle_ctx *oracle_create(int dim, int L, double J, double T, uint64_t seed)
{
    if (dim != 2 && dim != 3) return NULL;
    if (L < 2) return NULL;
    if (!(J >= 0.0) || !(T > 0.0) || !isfinite(J) || !isfinite(T)) return NULL;
    uint64_t N = 1;
    for (int k = 0; k < dim; ++k) {
        N *= (uint64_t)L;
        if (N > (1ull << 31)) return NULL;
    }
    oracle_ctx *h = (oracle_ctx *)calloc(1, sizeof(*h));
    if (!h) return NULL;
    h->dim = dim; h->L = L; h->N = N; h->J = J; h->T = T; h->seed = seed;
    h->thr = oracle_threshold(J, T);
    h->u = 0;
    h->s = (int8_t *)malloc(N);
    h->stack = (uint64_t *)malloc(N * sizeof(uint64_t));
    if (!h->s || !h->stack) { free(h->s); free(h->stack); free(h); return NULL; }
    for (uint64_t i = 0; i < N; ++i) h->s[i] = (int8_t)oracle_init_spin(seed, i);
    return h;
}

void oracle_destroy(oracle_ctx *h)
{
    if (!h) return;
    free(h->s); free(h->stack); free(h);
}

void oracle_get_spins(const oracle_ctx *h, int8_t *dst) { memcpy(dst, h->s, h->N); }
void oracle_set_spins(oracle_ctx *h, const int8_t *src) { memcpy(h->s, src, h->N); }
uint64_t oracle_get_threshold(const oracle_ctx *h) { return h->thr; }
uint64_t oracle_get_update_index(const oracle_ctx *h) { return h->u; }
void oracle_set_update_index(oracle_ctx *h, uint64_t u) { h->u = u; }

/* ----------------------------------------------------------------- update */

/* One single-cluster update, PAPER.md:42-48 steps (i)-(iv), with the flip at
 * the moment of joining (reading R3; PAPER.md:50 allows the timing) so that
 * "parallel with S_i and not a member before" is simply
 * s[j] == s0 (reading R2).  The list of PAPER.md:50 (counters ic, in) is a
 * LIFO stack here (reading R4).  Returns the cluster size. */
static uint64_t update_once(oracle_ctx *h)
{
    const uint64_t u = h->u;
    uint64_t top = 0, size = 0;
    /* (i) choose a site */
    uint64_t i0 = oracle_site_draw(h->seed, u, h->N);
    int8_t s0 = h->s[i0];
    h->s[i0] = (int8_t)-s0;
    h->stack[top++] = i0;
    size = 1;
    /* (ii)-(iv) */
    while (top > 0) {
        uint64_t i = h->stack[--top];
        for (int d = 0; d < h->dim; ++d) {
            for (int sign = +1; sign >= -1; sign -= 2) {
                uint64_t j = oracle_nbr(h->dim, h->L, i, d, sign);
                if (h->s[j] != s0) continue;
                uint64_t owner = (sign > 0) ? i : j;
                if (!oracle_bond_active(h->seed, u, owner, d, h->thr)) continue;
                h->s[j] = (int8_t)-s0;
                h->stack[top++] = j;
                ++size;
            }
        }
    }
    h->u = u + 1;   /* (v) */
    return size;
}

/* ------------------------------------------------------------ observables */

/* Reading R13 (PAPER.md:38 Eq. 2, :126): M = sum_i s_i and, in units of J,
 * E = - sum_i sum_{d<dim} s_i * s_{nbr(i,d,+)} (every bond once; for L = 2
 * the +d and -d neighbours coincide but are two bonds, both counted). */
void oracle_observables(const oracle_ctx *h, int64_t *E, int64_t *M)
{
    int64_t e = 0, m = 0;
    for (uint64_t i = 0; i < h->N; ++i) {
        m += h->s[i];
        for (int d = 0; d < h->dim; ++d)
            e -= (int64_t)h->s[i] * (int64_t)h->s[oracle_nbr(h->dim, h->L, i, d, +1)];
    }
    if (E) *E = e;
    if (M) *M = m;
}

/* n_updates updates; sizes (may be NULL) receives n_updates cluster sizes. */
int oracle_run(oracle_ctx *h, uint64_t n_updates, uint32_t *sizes)
{
    for (uint64_t k = 0; k < n_updates; ++k) {
        uint64_t c = update_once(h);
        if (sizes) sizes[k] = (uint32_t)c;
    }
    return 0;
}

/* Same, additionally logging E and M (full summation) after every update. */
int oracle_run_logged(oracle_ctx *h, uint64_t n_updates, uint32_t *sizes,
                      int64_t *E_log, int64_t *M_log)
{
    for (uint64_t k = 0; k < n_updates; ++k) {
        uint64_t c = update_once(h);
        if (sizes) sizes[k] = (uint32_t)c;
        oracle_observables(h, E_log ? &E_log[k] : NULL, M_log ? &M_log[k] : NULL);
    }
    return 0;
}

/* ----------------------------------------------------------------- moments */

/* Accumulated moments of a measured series and the Binder ratio.
 * PAPER.md:126 ("the measurement of energy and magnetization" after every
 * update; the "+ measurement" columns of Tables 1-2) and
 * PAPER.md:159-164 Eq. 3:  U(T) = 1 - <M^4> / (3 <M^2>^2),  averages over the
 * measured updates (the updates after the discarded ones).
 *
 * Definition, written out: over the n samples (E_k, M_k)
 *   out[0] = n              out[1] = sum E_k (two's complement)
 *   out[2] = sum |M_k|      out[3..4] = sum E_k^2  (low, high 64 bits)
 *   out[5..6] = sum M_k^2   out[7..8] = sum M_k^4  out[9] = 0 (reserved)
 * All sums are exact integers: M^4 reaches 2^96 at N = 2^24 spins, so the
 * second and fourth moments are kept in 128 bits.  `acc` continues an earlier
 * accumulation (acc may equal out; NULL starts from zero). */
void oracle_moments(uint64_t n, const int64_t *E, const int64_t *M, const uint64_t *acc, uint64_t out[10])
{
    uint64_t cnt = 0, sum_absM = 0;
    int64_t sum_E = 0;
    unsigned __int128 sum_E2 = 0, sum_M2 = 0, sum_M4 = 0;
    if (acc) {
        cnt = acc[0]; sum_E = (int64_t)acc[1]; sum_absM = acc[2];
        sum_E2 = ((unsigned __int128)acc[4] << 64) | acc[3];
        sum_M2 = ((unsigned __int128)acc[6] << 64) | acc[5];
        sum_M4 = ((unsigned __int128)acc[8] << 64) | acc[7];
    }
    for (uint64_t k = 0; k < n; ++k) {
        uint64_t absM = (uint64_t)(M[k] < 0 ? -M[k] : M[k]);
        uint64_t absE = (uint64_t)(E[k] < 0 ? -E[k] : E[k]);
        unsigned __int128 m2 = (unsigned __int128)absM * absM;
        cnt += 1;
        sum_E += E[k];
        sum_absM += absM;
        sum_E2 += (unsigned __int128)absE * absE;
        sum_M2 += m2;
        sum_M4 += m2 * m2;
    }
    out[0] = cnt; out[1] = (uint64_t)sum_E; out[2] = sum_absM;
    out[3] = (uint64_t)sum_E2; out[4] = (uint64_t)(sum_E2 >> 64);
    out[5] = (uint64_t)sum_M2; out[6] = (uint64_t)(sum_M2 >> 64);
    out[7] = (uint64_t)sum_M4; out[8] = (uint64_t)(sum_M4 >> 64);
    out[9] = 0;
}

/* Eq. 3 from the accumulated sums:
 * U = 1 - (S4/n) / (3 (S2/n)^2) = 1 - n S4 / (3 S2^2), in long double.
 * Returns NaN when no sample or S2 = 0. */
double oracle_binder(const uint64_t moments[10])
{
    long double n = (long double)moments[0];
    long double s2 = (long double)moments[6] * 18446744073709551616.0L + (long double)moments[5];
    long double s4 = (long double)moments[8] * 18446744073709551616.0L + (long double)moments[7];
    if (moments[0] == 0 || s2 == 0.0L) return (double)NAN;
    return (double)(1.0L - (n * s4) / (3.0L * s2 * s2));
}
