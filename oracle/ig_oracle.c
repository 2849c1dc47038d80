/* ORACLE - test infrastructure only. Plain, slow, fp64 CPU statement of what the
 * gridding path computes. Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may use it. It shares no code with the
 * CUDA path under paper_1403_4209_b200/csrc/.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC ig_oracle.c -o libig_oracle.so -lm
 *
 * What follows the paper (PAPER.md line : section/equation):
 *   orc_index : record -> (cell, sub-cell offset, w-plane, conj flag, on-grid)
 *               :1076-1091 sec 4.3.2 eq 4.1-4.2 (cell / delta-u rule),
 *               :546-564 sec 2.1.3 eq 2.11-2.13 (nearest oversampled sample),
 *               :633,:1068 (planes spaced in sqrt(w)), :1416-1427 eq 4.10 (conj
 *               trick for w<0), :1278,:1414 (records off the grid are dropped).
 *               Readings 1-4 of DESIGN.md fix what the paper leaves open.
 *   orc_grid  : grid[Y+ty][X+tx][pol] += eps*V * C_w(tap), :1266-1293 sec 4.4.2
 *               eq 4.4a/b; normaliser eq 4.5 with zeta of eq 4.3 (:1095);
 *               statistics eq 4.17 (:1552-1572).
 * Parity pins: tests/test_oracle_*.py (none of them re-use this file's formulas).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_C_M_S 299792458.0

/* floor division for possibly negative numerators */
static int64_t floordiv64(int64_t a, int64_t b) {
    int64_t q = a / b;
    if ((a % b != 0) && ((a < 0) != (b < 0))) q -= 1;
    return q;
}

/* The two scale constants of the index computation, written out once so that the
 * order of the fp64 operations is part of the contract (include/ig.h repeats it):
 *   du = 1/(N*cell_rad);  ku = beta/(c*du);  kw = (P-1)^2/(c*w_max). */
void orc_constants(int grid_n, double cell_rad, int beta, int n_wplanes, double w_max,
                   double *ku, double *kw) {
    double du = 1.0 / ((double)grid_n * cell_rad);
    *ku = (double)beta / (ORC_C_M_S * du);
    double pm1 = (double)(n_wplanes - 1);
    *kw = (n_wplanes > 1 && w_max > 0.0) ? (pm1 * pm1) / (ORC_C_M_S * w_max) : 0.0;
}

/* Per record (row r, channel c) in INPUT order, index r*nchan+c:
 *   X,Y      centre cell (pixel N/2 is u=v=0, :1319-1321)
 *   off_u/v  sub-cell offset in oversampled samples, in (-beta/2, beta/2]
 *   plane    w-plane, nearest in sqrt(w)
 *   flags    bit0 = conjugated (w<0), bit1 = whole footprint on the grid
 * A record with a non-finite coordinate (NaN or inf in u, v or w) is off the grid. */
void orc_index(int64_t nrow, int nchan, const double *uvw_m, const double *freqs_hz,
               int grid_n, double cell_rad, int beta, int n_wplanes, double w_max,
               const int32_t *support, int32_t *X, int32_t *Y, int32_t *off_u,
               int32_t *off_v, int32_t *plane, int32_t *flags) {
    double ku, kw;
    orc_constants(grid_n, cell_rad, beta, n_wplanes, w_max, &ku, &kw);
    const int64_t half_up = (beta + 1) / 2; /* ceil(beta/2) */
    for (int64_t r = 0; r < nrow; ++r) {
        double um = uvw_m[3 * r], vm = uvw_m[3 * r + 1], wm = uvw_m[3 * r + 2];
        int conj = wm < 0.0; /* eq 4.10: grid (-u,-v,-w) with conj(V) */
        if (conj) { um = -um; vm = -vm; wm = -wm; }
        for (int c = 0; c < nchan; ++c) {
            double nu = freqs_hz[c];
            double fu = (um * nu) * ku; /* (u/lambda) * beta/du, eq 1.7 + eq 2.11 */
            double fv = (vm * nu) * ku;
            int64_t k = r * nchan + c;
            if (!(isfinite(fu) && isfinite(fv) && isfinite(wm * nu))) {
                /* a non-finite coordinate has no cell (reading 20): the record is dropped like one
                 * whose footprint leaves the grid (:1278); its tuple is all zero apart from the conj bit */
                X[k] = 0; Y[k] = 0; off_u[k] = 0; off_v[k] = 0; plane[k] = 0; flags[k] = conj;
                continue;
            }
            int64_t U = (int64_t)ceil(fu - 0.5); /* nearest sample, ties to -inf */
            int64_t V = (int64_t)ceil(fv - 0.5);
            int64_t x = floordiv64(U + half_up - 1, beta); /* eq 4.2: -du/2 < delta <= du/2 */
            int64_t y = floordiv64(V + half_up - 1, beta);
            int64_t ou = U - x * beta, ov = V - y * beta;
            int64_t p = 0;
            if (n_wplanes > 1) {
                double sp = floor(sqrt((wm * nu) * kw) + 0.5);
                p = sp >= (double)(n_wplanes - 1) ? n_wplanes - 1 : (int64_t)sp;
            }
            int64_t h = (support[p] - 1) / 2;
            int64_t Xc = x + grid_n / 2, Yc = y + grid_n / 2;
            int on = (Xc - h >= 0) && (Xc + h <= grid_n - 1) && (Yc - h >= 0) && (Yc + h <= grid_n - 1);
            /* clamp far-off cells so they fit int32; they are off-grid anyway */
            if (Xc < -(1 << 30)) Xc = -(1 << 30);
            if (Xc > (1 << 30)) Xc = (1 << 30);
            if (Yc < -(1 << 30)) Yc = -(1 << 30);
            if (Yc > (1 << 30)) Yc = (1 << 30);
            X[k] = (int32_t)Xc; Y[k] = (int32_t)Yc;
            off_u[k] = (int32_t)ou; off_v[k] = (int32_t)ov;
            plane[k] = (int32_t)p;
            flags[k] = conj | (on << 1);
        }
    }
}

/* Gridding by definition (eq 4.4). bank: fp64 complex, plane p starts at
 * bank_off[p] (in complex elements), laid out [ov][ou][ty][tx] with
 * ov,ou = off + ceil(beta/2) - 1 in [0,beta) (:1100-1108 layout C-1).
 * grid: fp64 complex [N][N][npol], ADDED to. norm[npol] ADDED to.
 * stats[0] += gridded records, [1] += dropped records, [2] += sum S^2 * npol.
 * A record is gridded iff on-grid and at least one polarisation weight != 0
 * (:1315 all-flagged records are dropped; weight 0 plays the flag's role).
 * Threads own bands of grid rows: no atomics, deterministic for a given input. */
void orc_grid(int64_t nrow, int nchan, int npol, const float *vis /*[nrow][nchan][npol][2]*/,
              const float *wt /*[nrow][nchan][npol]*/, const int32_t *X, const int32_t *Y,
              const int32_t *off_u, const int32_t *off_v, const int32_t *plane,
              const int32_t *flags, int grid_n, int beta, const int32_t *support,
              const int64_t *bank_off, const double *bank, double *grid, double *norm,
              int64_t *stats) {
    const int64_t nrec = nrow * nchan;
    const int shift = (beta + 1) / 2 - 1;
    int64_t gridded = 0, dropped = 0, updates = 0;
    double nsum[4] = {0, 0, 0, 0};
    /* pass 1: counters and normaliser (serial, fixed order) */
    for (int64_t k = 0; k < nrec; ++k) {
        int any = 0;
        for (int q = 0; q < npol; ++q) any |= (wt[k * npol + q] != 0.0f);
        if (!(flags[k] & 2) || !any) { dropped++; continue; }
        int p = plane[k], S = support[p];
        const double *K = bank + 2 * (bank_off[p] + ((int64_t)(off_v[k] + shift) * beta + (off_u[k] + shift)) * S * S);
        double zeta = 0.0; /* eq 4.3 */
        for (int t = 0; t < S * S; ++t) zeta += K[2 * t];
        for (int q = 0; q < npol; ++q) nsum[q] += (double)wt[k * npol + q] * zeta; /* eq 4.5 */
        gridded++;
        updates += (int64_t)S * S * npol;
    }
    /* pass 2: the grid, banded by rows */
#pragma omp parallel
    {
        int nt = 1, tid = 0;
#ifdef _OPENMP
        nt = omp_get_num_threads(); tid = omp_get_thread_num();
#endif
        int y0 = (int)((int64_t)grid_n * tid / nt), y1 = (int)((int64_t)grid_n * (tid + 1) / nt);
        for (int64_t k = 0; k < nrec; ++k) {
            if (!(flags[k] & 2)) continue;
            int p = plane[k], S = support[p], h = (S - 1) / 2;
            int Yc = Y[k], Xc = X[k];
            if (Yc + h < y0 || Yc - h >= y1) continue;
            int any = 0;
            double a_re[4], a_im[4];
            for (int q = 0; q < npol; ++q) {
                double w = (double)wt[k * npol + q];
                any |= (w != 0.0);
                a_re[q] = w * (double)vis[2 * (k * npol + q)];
                a_im[q] = w * (double)vis[2 * (k * npol + q) + 1];
                if (flags[k] & 1) a_im[q] = -a_im[q]; /* eq 4.16b */
            }
            if (!any) continue;
            const double *K = bank + 2 * (bank_off[p] + ((int64_t)(off_v[k] + shift) * beta + (off_u[k] + shift)) * S * S);
            for (int ty = -h; ty <= h; ++ty) {
                int gy = Yc + ty;
                if (gy < y0 || gy >= y1) continue;
                for (int tx = -h; tx <= h; ++tx) {
                    const double *kv = K + 2 * ((int64_t)(ty + h) * S + (tx + h));
                    double *g = grid + 2 * (((int64_t)gy * grid_n + (Xc + tx)) * npol);
                    for (int q = 0; q < npol; ++q) {
                        g[2 * q] += a_re[q] * kv[0] - a_im[q] * kv[1];
                        g[2 * q + 1] += a_re[q] * kv[1] + a_im[q] * kv[0];
                    }
                }
            }
        }
    }
    for (int q = 0; q < npol; ++q) norm[q] += nsum[q];
    stats[0] += gridded; stats[1] += dropped; stats[2] += updates;
}

/* measurement infrastructure only: thread count of the next orc_grid calls (0 = the OpenMP default) */
void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int orc_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
