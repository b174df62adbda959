/*
 * ising_enum.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Brute-force enumeration of every state of a small periodic Ising lattice
 * (Eq. 2: H = -J sum_<ij> S_i S_j, periodic boundaries).
 * It is the pin for the oracle's sampler: Boltzmann averages computed from
 * the joint density of states g(E, M) returned here are what a correct Wolff
 * chain must reproduce within statistical error.
 *
 * Deliberately independent of wolff_oracle.c: own neighbour arithmetic
 * (explicit coordinates), no Philox, no shared helper.  Walks the 2^N states
 * in Gray-code order, updating E and M by the single flipped spin.
 *
 * g is indexed [ (E + dim*N) * (2N+1) + (M + N) ], E in units of J.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

int ising_enum_joint_dos(int dim, int L, uint64_t *g /* (2*dim*N+1)*(2N+1) */)
{
    if (dim < 1 || dim > 3 || L < 2) return -1;
    int N = 1;
    for (int k = 0; k < dim; ++k) N *= L;
    if (N > 30) return -1;

    /* neighbour table with multiplicity: 2*dim entries per site */
    int (*nb)[6] = malloc(sizeof(int[6]) * (size_t)N);
    if (!nb) return -2;
    for (int i = 0; i < N; ++i) {
        int c[3] = {0, 0, 0};
        int rest = i;
        for (int k = 0; k < dim; ++k) { c[k] = rest % L; rest /= L; }
        for (int d = 0; d < dim; ++d) {
            for (int pm = 0; pm < 2; ++pm) {
                int cc[3] = { c[0], c[1], c[2] };
                cc[d] = pm ? (c[d] + L - 1) % L : (c[d] + 1) % L;
                int j = 0;
                for (int k = dim - 1; k >= 0; --k) j = j * L + cc[k];
                nb[i][2 * d + pm] = j;
            }
        }
    }

    const int nE = 2 * dim * N + 1, nM = 2 * N + 1;
    memset(g, 0, sizeof(uint64_t) * (size_t)nE * (size_t)nM);

    int8_t s[32];
    for (int i = 0; i < N; ++i) s[i] = -1;       /* Gray code 0: all spins down */
    int E = -dim * N, M = -N;                     /* every one of dim*N bonds satisfied */
    const uint64_t total = 1ull << N;
    for (uint64_t t = 0;; ) {
        g[(size_t)(E + dim * N) * (size_t)nM + (size_t)(M + N)] += 1;
        if (++t == total) break;
        int k = __builtin_ctzll(t);               /* Gray code: flip bit ctz(t) */
        int sum = 0;
        for (int q = 0; q < 2 * dim; ++q) sum += s[nb[k][q]];
        E += 2 * s[k] * sum;                      /* E = -sum s_i s_j over bonds */
        M -= 2 * s[k];
        s[k] = (int8_t)-s[k];
    }
    free(nb);
    return 0;
}
