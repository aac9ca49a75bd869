/*
 * TRED hot-path ORACLE (C part) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 restatement of PAPER.md (arxiv 2602.12052) Sec. II-C/II-D.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this.  It shares no code with the CUDA path.
 *
 *   tred_o_q            Eq. (10) with the exponent read as
 *                       exp(-B/(2 Delta^2)) (reading G1) and the
 *                       point-like branch of PAPER.md:L148.
 *   tred_o_effq         Eq. (9): scatter of
 *                       w_lmn * q(node) * u_lmn,rst onto grid points.
 *   tred_o_conv_direct  Eq. (12) as a direct sum, no FFT.
 *
 * Loops are in the paper's order (segment -> cuboid -> node (l,m,n) ->
 * neighbour (r,s,t)); there is no blocking, fusion or reordering.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 *
 * Pins (tests/test_oracle_*.py): scipy quadrature of the defining line (x)
 * Gaussian integral, total charge, n=1 closed form, adjoint/interpolation
 * identity, impulse response, FFT-vs-direct, shift equivariance, linearity.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* Charge density of one diffused segment at pos = (x, y, t).
 * p0, p1: segment ends (x [mm], y [mm], arrival time [us]); sig: (sx, sy, st);
 * Qp: surviving electrons.  Result: electrons / (mm^2 us).             */
double tred_o_q(const double *p0, const double *p1, const double *sig,
                double Qp, int point_like, const double *pos)
{
    if (point_like) {                       /* PAPER.md:L148, midpoint Gaussian */
        double g = Qp;
        for (int a = 0; a < 3; ++a) {
            double m = 0.5 * (p0[a] + p1[a]);
            double u = (pos[a] - m) / sig[a];
            g *= exp(-0.5 * u * u) / (sqrt(2.0 * M_PI) * sig[a]);
        }
        return g;
    }
    /* a = d^T S^-1 d, b = d^T S^-1 r, c = r^T S^-1 r with d = p1-p0, r = pos-p0.
     * Eq. (10): Delta = sx sy st sqrt(a); B/Delta^2 = c - b^2/a (Lagrange);
     * -A_1/(sqrt2 Delta sx sy st) = b/sqrt(2a); A_2/(...) = (a-b)/sqrt(2a).      */
    double a = 0.0, b = 0.0, c = 0.0;
    for (int k = 0; k < 3; ++k) {
        double d = p1[k] - p0[k], r = pos[k] - p0[k], s2 = sig[k] * sig[k];
        a += d * d / s2;
        b += d * r / s2;
        c += r * r / s2;
    }
    double Delta = sig[0] * sig[1] * sig[2] * sqrt(a);
    double ex = exp(-0.5 * (c - b * b / a));
    double er = erf((a - b) / sqrt(2.0 * a)) + erf(b / sqrt(2.0 * a));
    return Qp / (4.0 * M_PI * Delta) * ex * er;
}

typedef struct {
    int64_t NG[3];      /* fine grid points per axis (x, y, t)              */
    int64_t B[3];       /* block shape                                       */
    int64_t NB[3];      /* blocks per axis = ceil(NG/B)                      */
    double  org[3];     /* origin_x, origin_y, t_origin                      */
    double  h[3];       /* spacing hx, hy, dt                                */
} tred_o_grid;

static inline int64_t fdiv(int64_t a, int64_t b) { /* floor division, b > 0 */
    int64_t q = a / b;
    return (a % b != 0 && a < 0) ? q - 1 : q;
}

/* Eq. (9).  For every segment, every cuboid c in its bbox [lo,hi]^3, every GL
 * node (l,m,n): position (c + 1/2 + xi/2) h, weight w h/2 per axis, charge q;
 * scatter with u_{l,r} (r = -1,0,+1 stored at index r+1) to grid point c + r.
 * Grid point (i,j,k) is the CENTRE of cuboid (i,j,k) (reading G4).
 * Points outside the grid or in a block whose slot is < 0 are dropped.
 * blockslot[(bt*NBx + bx)*NBy + by] -> payload slot; payload [slot][Bx][By][Bt]. */
void tred_o_effq(const tred_o_grid *g, int64_t nseg,
                 const double *p0 /*[nseg][3]*/, const double *p1, const double *sig /*[nseg][3]*/,
                 const double *Qp, const int32_t *point_like,
                 const int64_t *lo /*[nseg][3]*/, const int64_t *hi,
                 int n, const double *xi, const double *w, const double *u /*[n][3]*/,
                 const int64_t *blockslot, double *payload)
{
    const int64_t Bx = g->B[0], By = g->B[1], Bt = g->B[2];
    #pragma omp parallel for schedule(dynamic, 4)
    for (int64_t s = 0; s < nseg; ++s) {
        const double *a0 = p0 + 3 * s, *a1 = p1 + 3 * s, *sg = sig + 3 * s;
        for (int64_t cx = lo[3*s+0]; cx <= hi[3*s+0]; ++cx)
        for (int64_t cy = lo[3*s+1]; cy <= hi[3*s+1]; ++cy)
        for (int64_t ct = lo[3*s+2]; ct <= hi[3*s+2]; ++ct) {
            for (int l = 0; l < n; ++l)
            for (int m = 0; m < n; ++m)
            for (int nn = 0; nn < n; ++nn) {
                double pos[3];
                pos[0] = g->org[0] + ((double)cx + 0.5 + 0.5 * xi[l])  * g->h[0];
                pos[1] = g->org[1] + ((double)cy + 0.5 + 0.5 * xi[m])  * g->h[1];
                pos[2] = g->org[2] + ((double)ct + 0.5 + 0.5 * xi[nn]) * g->h[2];
                double wq = (w[l] * 0.5 * g->h[0]) * (w[m] * 0.5 * g->h[1]) * (w[nn] * 0.5 * g->h[2])
                          * tred_o_q(a0, a1, sg, Qp[s], point_like[s], pos);
                for (int r = -1; r <= 1; ++r)
                for (int q = -1; q <= 1; ++q)
                for (int t = -1; t <= 1; ++t) {
                    double coef = u[3*l + r + 1] * u[3*m + q + 1] * u[3*nn + t + 1];
                    if (coef == 0.0) continue;
                    int64_t i = cx + r, j = cy + q, k = ct + t;
                    if (i < 0 || j < 0 || k < 0 || i >= g->NG[0] || j >= g->NG[1] || k >= g->NG[2]) continue;
                    int64_t bx = i / Bx, by = j / By, bt = k / Bt;
                    int64_t slot = blockslot[(bt * g->NB[0] + bx) * g->NB[1] + by];
                    if (slot < 0) continue;
                    double *dst = payload + ((slot * Bx + (i - bx * Bx)) * By + (j - by * By)) * Bt + (k - bt * Bt);
                    #pragma omp atomic
                    *dst += wq * coef;
                }
            }
        }
    }
}

/* Eq. (12) as a direct sum (reading O5):
 *   I[px,py,t] = sum_{jx,jy} sum_{kx,ky=-H..H} sum_{tau<Tr}
 *                Qeff[(px-kx)S+jx, (py-ky)S+jy, t-tau] * R[jx,jy,kx+H,ky+H,tau]
 * for the pixels listed in pix (flat id px*Npy+py); out [npix][Nt].
 * Qeff is read from the block-sparse payload (zero where no block).       */
void tred_o_conv_direct(const tred_o_grid *g, int64_t S, int64_t H, int64_t Tr,
                        int64_t Npx, int64_t Npy,
                        const int64_t *blockslot, const double *payload,
                        const float *R, int64_t npix, const int64_t *pix, double *out)
{
    const int64_t Bx = g->B[0], By = g->B[1], Bt = g->B[2], Nt = g->NG[2];
    const int64_t K = 2 * H + 1;
    #pragma omp parallel for schedule(dynamic, 1)
    for (int64_t ip = 0; ip < npix; ++ip) {
        int64_t px = pix[ip] / Npy, py = pix[ip] % Npy;
        double *o = out + ip * Nt;
        for (int64_t t = 0; t < Nt; ++t) o[t] = 0.0;
        for (int64_t kx = -H; kx <= H; ++kx)
        for (int64_t ky = -H; ky <= H; ++ky) {
            int64_t cpx = px - kx, cpy = py - ky;       /* pixel holding the charge */
            if (cpx < 0 || cpy < 0 || cpx >= Npx || cpy >= Npy) continue;
            for (int64_t jx = 0; jx < S; ++jx)
            for (int64_t jy = 0; jy < S; ++jy) {
                int64_t i = cpx * S + jx, j = cpy * S + jy;
                int64_t bx = i / Bx, by = j / By;
                const float *r = R + ((((jx * S + jy) * K + (kx + H)) * K) + (ky + H)) * Tr;
                for (int64_t bt = 0; bt < g->NB[2]; ++bt) {
                    int64_t slot = blockslot[(bt * g->NB[0] + bx) * g->NB[1] + by];
                    if (slot < 0) continue;
                    const double *qv = payload + ((slot * Bx + (i - bx * Bx)) * By + (j - by * By)) * Bt;
                    for (int64_t tl = 0; tl < Bt; ++tl) {
                        double q = qv[tl];
                        if (q == 0.0) continue;
                        int64_t t = bt * Bt + tl;
                        int64_t tmax = (Nt - t < Tr) ? Nt - t : Tr;
                        for (int64_t tau = 0; tau < tmax; ++tau) o[t + tau] += q * (double)r[tau];
                    }
                }
            }
        }
    }
}

int tred_o_abi_version(void) { return 1; }
