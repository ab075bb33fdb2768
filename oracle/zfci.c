/*
 * ORACLE (test infrastructure, not product code): the dense determinant-basis Hamiltonian of Eq. (2)
 * for COMPLEX Hermitian spin-orbital integrals without spin selection rules -- the Hamiltonian "including spin-orbit
 * couplings" of PAPER.md:97 -- by the Slater-Condon rules.  This is the plain definition of the exact result that
 * oracle/zsigma.py is pinned to (tests/test_oracle_spinorbit.py); it is itself pinned to an independent Jordan-Wigner
 * construction (tests/fockdense.py).  Shares no code with the CUDA path.
 *
 * Determinants are bit strings over n spin orbitals, bit P set = a+_P present, creation operators in ascending
 * P order (DESIGN.md conventions).  h[n*n] and V[n^4] = <PQ||RS> are complex, interleaved (re, im) pairs.
 * H[bra][ket] = <bra| H |ket>.
 */
#include <complex.h>
#include <stdint.h>
#include <stddef.h>

static inline int zpopc(uint64_t x) { return __builtin_popcountll(x); }
static inline int zbelow(uint64_t d, int P) { return zpopc(d & ((1ULL << P) - 1)); }
static int z_ann(uint64_t *d, int P, int *sgn) {
    if (!((*d >> P) & 1)) return 0;
    if (zbelow(*d, P) & 1) *sgn = -*sgn;
    *d &= ~(1ULL << P);
    return 1;
}
static int z_cre(uint64_t *d, int P, int *sgn) {
    if ((*d >> P) & 1) return 0;
    if (zbelow(*d, P) & 1) *sgn = -*sgn;
    *d |= (1ULL << P);
    return 1;
}

static double complex zfci_element(uint64_t bra, uint64_t ket, int n, const double complex *h, const double complex *V) {
#define VV(p, q, r, s) V[(((size_t)(p) * n + (q)) * n + (r)) * n + (s)]
    uint64_t diff = bra ^ ket;
    int nd = zpopc(diff);
    if (nd == 0) {   /* sum_i h_ii + 1/2 sum_ij <ij||ij> */
        double complex e = 0.0;
        for (int i = 0; i < n; i++) if ((ket >> i) & 1) {
            e += h[i * n + i];
            for (int j = 0; j < n; j++) if ((ket >> j) & 1) e += 0.5 * VV(i, j, i, j);
        }
        return e;
    }
    if (nd == 2) {   /* ket -> bra replaces i by a:  phase * (h_ai + sum_j <aj||ij>) */
        int i = __builtin_ctzll(ket & diff), a = __builtin_ctzll(bra & diff);
        int lo = i < a ? i : a, hi = i < a ? a : i;
        uint64_t between = ket & (((1ULL << hi) - 1) & ~((1ULL << (lo + 1)) - 1));
        double ph = (zpopc(between) & 1) ? -1.0 : 1.0;
        double complex e = h[a * n + i];
        for (int j = 0; j < n; j++) if ((ket >> j) & 1) e += VV(a, j, i, j);
        return ph * e;
    }
    if (nd == 4) {   /* i<j -> a<b:  sign of a+_a a+_b a_j a_i on the ket times <ab||ij> */
        uint64_t from = ket & diff, to = bra & diff;
        int i = __builtin_ctzll(from), j = 63 - __builtin_clzll(from);
        int a = __builtin_ctzll(to), b = 63 - __builtin_clzll(to);
        uint64_t d = ket; int sgn = 1;
        z_ann(&d, i, &sgn); z_ann(&d, j, &sgn); z_cre(&d, b, &sgn); z_cre(&d, a, &sgn);
        return sgn * VV(a, b, i, j);
    }
    return 0.0;
#undef VV
}

void zfci_dense_h(const uint64_t *dets, int64_t ndet, int n, const double complex *h, const double complex *V, double complex *H) {
    for (int64_t i = 0; i < ndet; i++)
        for (int64_t j = 0; j < ndet; j++)
            H[i * ndet + j] = zfci_element(dets[i], dets[j], n, h, V);
}
