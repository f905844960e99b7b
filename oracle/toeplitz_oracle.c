/* CPU oracle helper (TEST INFRASTRUCTURE ONLY): the O(n^2) Toeplitz product of Eq. 4,
 *     (T x)_{c,m} = sum_{m'} coef_{m-m'} x_{c,m'},
 * written as the plain six-deep loop.  No FFT, no blocking, no reordering; OpenMP only splits the
 * independent output harmonics across host cores.  Pinned to the numpy statement
 * oracle/gsm_oracle.py:toeplitz_matvec in tests/test_oracle_pins.py.
 *
 * Layouts (interleaved re,im doubles): coef[(2N1-1)][(2N2-1)][(2N3-1)] indexed d_a + N_a - 1;
 * x, y[3][N1][N2][N3].
 */
#include <complex.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void toeplitz_matvec_c(const double complex* coef, const double complex* x, double complex* y,
                       int N1, int N2, int N3) {
    const long D2 = 2 * N2 - 1, D3 = 2 * N3 - 1;
    const long n = (long)N1 * N2 * N3;
#pragma omp parallel for collapse(2) schedule(static)
    for (int i1 = 0; i1 < N1; ++i1)
        for (int i2 = 0; i2 < N2; ++i2)
            for (int i3 = 0; i3 < N3; ++i3) {
                double complex s0 = 0, s1 = 0, s2 = 0;
                for (int j1 = 0; j1 < N1; ++j1)
                    for (int j2 = 0; j2 < N2; ++j2) {
                        const double complex* cr =
                            coef + ((long)(i1 - j1 + N1 - 1) * D2 + (i2 - j2 + N2 - 1)) * D3 + (i3 + N3 - 1);
                        const double complex* xr = x + ((long)j1 * N2 + j2) * N3;
                        for (int j3 = 0; j3 < N3; ++j3) {
                            const double complex cc = cr[-j3];
                            s0 += cc * xr[j3];
                            s1 += cc * xr[n + j3];
                            s2 += cc * xr[2 * n + j3];
                        }
                    }
                const long o = ((long)i1 * N2 + i2) * N3 + i3;
                y[o] = s0;
                y[n + o] = s1;
                y[2 * n + o] = s2;
            }
}
