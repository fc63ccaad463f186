/* Oracle, pin P6 and the timed CPU baseline: a literal transcription of the paper's Algorithm 1,
 * "Action of spin operator S on state |Psi>", on the <bits, coeff> encoding of
 * PAPER.md:257-267.  TEST INFRASTRUCTURE ONLY -- never linked into the CUDA library.
 *
 *   for 0 <= m < 2^L:
 *     for each <bits, coeff> in S:
 *       n <- m; minus <- false
 *       for each i-th non-zero bit of bits:             (scanned from the LSB)
 *         if i is even: flip qubit i/2 of n             (DESIGN.md R-ALG1-BIT)
 *         else if qubit i/2 of n is set: flip minus
 *       if minus is false: Phi[m] += coeff*Psi[n]
 *       else:              Phi[m] -= coeff*Psi[n]       (the missing `else` is R-ALG1-ELSE)
 *
 * The paper's own CPU fallback is this algorithm under OpenMP, hence the one pragma.
 * Vectors are interleaved (re, im) doubles.  Rows [m_begin, m_end) of Phi are written to phi[0..].
 */
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int alg1_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void alg1_apply(int L, int64_t n_tuples, const uint64_t *bits, const double *coeff,
                const double *psi, double *phi, uint64_t m_begin, uint64_t m_end)
{
    (void)L;
    int64_t rows = (int64_t)(m_end - m_begin);
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < rows; ++r) {
        uint64_t m = m_begin + (uint64_t)r;
        double acc_re = 0.0, acc_im = 0.0;
        for (int64_t s = 0; s < n_tuples; ++s) {
            uint64_t n = m;
            int minus = 0;
            for (uint64_t rest = bits[s]; rest; rest &= rest - 1) {
                int i = __builtin_ctzll(rest);
                if ((i & 1) == 0)
                    n ^= (uint64_t)1 << (i >> 1);
                else if ((n >> (i >> 1)) & 1)
                    minus = !minus;
            }
            double cr = coeff[2 * s], ci = coeff[2 * s + 1];
            double pr = psi[2 * n], pi = psi[2 * n + 1];
            double tr = cr * pr - ci * pi, ti = cr * pi + ci * pr;
            if (!minus) { acc_re += tr; acc_im += ti; }
            else        { acc_re -= tr; acc_im -= ti; }
        }
        phi[2 * r] = acc_re;
        phi[2 * r + 1] = acc_im;
    }
}
