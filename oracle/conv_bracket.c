/* oracle/conv_bracket.c -- TEST INFRASTRUCTURE ONLY (part of the fp64 CPU oracle).
 *
 * Plain-C transcription of gx_oracle.bracket_convolution: the *definition* of the
 * dealiased Poisson bracket in k space (App. D Eq. D1 line 1,
 * with the 2/3-rule truncation of line 655):
 *
 *   C_k[chi,g] = sum_{p+q=k; p,q in K+-} (p_x q_y - p_y q_x) chi_p g_q ,   k in K
 *
 * K   = { (a,b) : |a| <= K, 0 <= b <= Q }   compact set, stored [nakx][naky] with the kx
 *       integers in the order 0..K,-K..-1 and interleaved (re,im) doubles;
 * K+- = K extended to b < 0 by the reality condition f(-p) = conj f(p).
 *
 * No blocking, no reordering beyond the loop nest below; OpenMP only distributes the
 * independent output modes k.  Shares nothing with the CUDA path.
 */
#include <complex.h>
#include <stdlib.h>

static inline double complex ext(const double complex *F, int nakx, int naky, int a, int b)
{
    /* value of the reality-extended field at integer mode (a,b), |a|<=K, |b|<=Q */
    if (b < 0) {
        int ia = (-a >= 0) ? -a : -a + nakx;
        return conj(F[ia * naky + (-b)]);
    }
    int ia = (a >= 0) ? a : a + nakx;
    return F[ia * naky + b];
}

void gxo_bracket_convolution(int nakx, int naky, double dkx, double dky,
                             const double complex *chi, const double complex *g,
                             double complex *out)
{
    const int K = (nakx - 1) / 2, Q = naky - 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int i = 0; i < nakx; ++i) {
        for (int kb = 0; kb < naky; ++kb) {
            const int ka = (i <= K) ? i : i - nakx;
            double complex acc = 0.0;
            for (int pa = -K; pa <= K; ++pa) {
                const int qa = ka - pa;
                if (abs(qa) > K) continue;
                for (int pb = -Q; pb <= Q; ++pb) {
                    const int qb = kb - pb;
                    if (abs(qb) > Q) continue;
                    const double px = dkx * pa, py = dky * pb, qx = dkx * qa, qy = dky * qb;
                    acc += (px * qy - py * qx) * ext(chi, nakx, naky, pa, pb) * ext(g, nakx, naky, qa, qb);
                }
            }
            out[i * naky + kb] = acc;
        }
    }
}
