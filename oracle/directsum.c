/* Matrix-free direct-sum product with the slope-slope covariance (oracle, fp64).
 * TEST INFRASTRUCTURE ONLY: shares no code with the CUDA path.
 *
 * q[i,a,p] = sum_{j,b} sum_{p'} theta[i,a,j,b](p' - p) x[j,b,p']
 * which is W_s Sigma_ss W_s^T x written out entry by entry (Eq.29,
 * Eq.34) with each Theta_{p,q} entry looked up in its (2n-1)^2 generator
 * (L150): no FFT, no reordering.  p, p' run over the valid subapertures only.
 *
 * theta : [C][C][L][L] doubles, C = 2*N channels, L = 2n-1, index (ly+n-1, lx+n-1),
 *         lag = input - output position on the n x n grid.
 * ix,iy : [nv] grid coordinates of the valid subapertures.
 * x, q  : [C][nv].
 */
#include <stddef.h>

void directsum_css(const double *theta, int C, int n, int nv,
                   const int *ix, const int *iy, const double *x, double *q)
{
    const int L = 2 * n - 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int co = 0; co < C; ++co) {
        for (int p = 0; p < nv; ++p) {
            double acc = 0.0;
            const int px = ix[p], py = iy[p];
            for (int ci = 0; ci < C; ++ci) {
                const double *g = theta + ((size_t)co * C + ci) * L * L;
                const double *xv = x + (size_t)ci * nv;
                double s = 0.0;
                for (int pp = 0; pp < nv; ++pp) {
                    const int lx = ix[pp] - px + (n - 1);
                    const int ly = iy[pp] - py + (n - 1);
                    s += g[(size_t)ly * L + lx] * xv[pp];
                }
                acc += s;
            }
            q[(size_t)co * nv + p] = acc;
        }
    }
}

/* Same entry-by-entry product for the phase-slope generators of one layer:
 * g[p'] = sum_{c} sum_{q} xi[c](q - p') x[c,q],  p' on the full n' x n' grid,
 * lag index (ly + n'-1, lx + n'-1), L = n' + n - 1  (Eq.32 L290 without the FFT). */
void directsum_cos_layer(const double *xi, int C, int n, int np_, int nv,
                         const int *ix, const int *iy, const double *x, double *g)
{
    const int L = np_ + n - 1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int py = 0; py < np_; ++py) {
        for (int px = 0; px < np_; ++px) {
            double acc = 0.0;
            for (int c = 0; c < C; ++c) {
                const double *t = xi + (size_t)c * L * L;
                const double *xv = x + (size_t)c * nv;
                double s = 0.0;
                for (int q = 0; q < nv; ++q) {
                    const int lx = ix[q] - px + (np_ - 1);
                    const int ly = iy[q] - py + (np_ - 1);
                    s += t[(size_t)ly * L + lx] * xv[q];
                }
                acc += s;
            }
            g[(size_t)py * np_ + px] = acc;
        }
    }
}
