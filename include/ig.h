/* ig.h - C ABI of the B200 convolutional gridder with W-projection.
 *
 * The operations are the ones the thesis states (citations are PAPER.md line :
 * section / equation; "reading k" = DESIGN.md table of readings):
 *   ig_build_wkernels  Algorithm 4.1 (:1122-1149), bank layout :1100-1108, eq 4.1-4.3
 *   ig_grid            WImager, eq 4.4a/b and 4.5 (:1266-1293); record preparation
 *                      sec 4.4.5 (:1385-1444); ordering :714, :1613-1646; plan eq 4.8
 *   ig_finalize        Algorithm 4.6 (:1664-1676), eq 2.9 (:523), eq 2.13 (:561-564)
 *   ig_get_stats       eq 4.17 (:1552-1572), metric definitions sec 5.3 (:1757-1779)
 *
 * Conventions
 *  - Plain C, no torch types. Every pointer says host or dev(ice). The caller owns
 *    ALL buffers and the CUDA stream; the library never allocates or frees device
 *    memory (PyTorch does, in the Python binding and in the tests).
 *  - Every call returns an ig_status; nothing throws or aborts across the ABI.
 *    ig_last_error() gives the text of the last failure on that context.
 *  - Work is enqueued on the bound stream and calls return without waiting, except
 *    the calls that hand back host data (ig_finalize's normaliser, ig_get_stats,
 *    ig_debug_*), which synchronise the stream first.
 *  - State machine: create -> bind -> build_wkernels (or debug_set_wkernels) ->
 *    grid* -> finalize. A call out of order returns IG_ESTATE.
 *  - One context = one grid (thesis: one WImager instance per grid, :1120).
 *  - There is no CPU fallback anywhere: without a CUDA device every compute call
 *    returns IG_ECUDA.
 */
#ifndef IG_H
#define IG_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ig_ctx ig_ctx; /* opaque */

typedef enum {
    IG_OK = 0,
    IG_EINVAL = 1,      /* bad argument */
    IG_ESTATE = 2,      /* call out of order */
    IG_ECUDA = 3,       /* CUDA runtime error (text in ig_last_error) */
    IG_ENOMEM = 4,      /* a caller-provided buffer is too small */
    IG_EUNSUPPORTED = 5 /* valid request this build does not implement */
} ig_status;

#define IG_C_M_S 299792458.0 /* speed of light used for metres -> wavelengths */
#define IG_MAX_SUPPORT 511   /* largest support the thesis sweeps (:1785-1789); record headers carry it in 9 bits */

/* Create a context. No device work.
 *   grid_n        grid side N, even, 16..32768
 *   cell_rad      image pixel size in radians; uv cell du = 1/(N*cell_rad) wavelengths
 *   n_wplanes     P >= 1 w-planes spaced in sqrt(w) (:633,:1068); 1 = plain gridding
 *   oversampling  beta in 1..16 (eq 2.11 :548)
 *   max_support   largest kernel support, odd, 3..IG_MAX_SUPPORT (the thesis's heavy configuration needs
 *                 349, :1924); a valid odd support above IG_MAX_SUPPORT returns IG_EUNSUPPORTED
 *   n_pol         1, 2 or 4 polarisations (:1025,:1377)                           */
ig_status ig_create(ig_ctx** out, int grid_n, double cell_rad, int n_wplanes, int oversampling,
                    int max_support, int n_pol);
void ig_destroy(ig_ctx* ctx);
const char* ig_last_error(const ig_ctx* ctx);

/* Bytes of the uv-grid: N*N*n_pol complex64. Layout (reading 13): n_pol 1 or 2: [y][x][pol][re,im]
 * ("multi-polarised pixel", :1319); n_pol 4: two planes of polarisation pairs, [pair][y][x][2][re,im]
 * with pol = 2*pair + k, so that a pixel commit is two 16-byte vector reductions and neighbouring
 * pixels share L2 sectors. Pixel (N/2,N/2) is u=v=0. */
size_t ig_grid_bytes(const ig_ctx* ctx);
/* Bytes of work_dev that one ig_grid call of (nrow, nchan) needs, for the context as it stands: the plan arrays and
 * the entry area of the gather gridder (80 B per record at 4 polarisations, the largest part) are counted only when a
 * record can reach it, i.e. not when the installed support table stays below ig_set_gather_min_support's threshold
 * (before a table is installed, max_support decides); with per-channel grids the plan arrays grow with nchan. Ask again
 * after changing the table, the threshold or the per-channel switch; ig_grid checks the bound size and returns
 * IG_ENOMEM if short. */
size_t ig_workspace_bytes(const ig_ctx* ctx, long long nrow, int nchan);
/* Bytes of the kernel bank for this support table [n_wplanes] (host; NULL = upper
 * bound with every plane at max_support). */
size_t ig_bank_bytes(const ig_ctx* ctx, const int* support_table);
/* Bytes of work_dev that ig_finalize needs. */
size_t ig_finalize_workspace_bytes(const ig_ctx* ctx);

/* Bind caller-owned device memory and the stream.
 *   grid_dev   dev, ig_grid_bytes(); ig_grid ADDS into it, the caller zeroes it
 *   work_dev   dev, 256-byte aligned scratch, contents undefined between calls
 *   bank_dev   dev, holds the kernel bank from ig_build_wkernels on; read-only after
 *   cuda_stream  a cudaStream_t (0 = default stream)
 * May be called again to change buffers; the bank must then be rebuilt if bank_dev moved. */
ig_status ig_bind(ig_ctx* ctx, void* grid_dev, size_t grid_bytes, void* work_dev, size_t work_bytes,
                  void* bank_dev, size_t bank_bytes, void* cuda_stream);

/* Build the bank on the device (Algorithm 4.1 as a direct DFT, reading 5):
 *   C_p = DFT_{beta*n zero padded}( psi(l) psi(m) exp(+j 2 pi w_p (sqrt(1-l^2-m^2)-1)) ) / A,
 *   w_p = w_max (p/(P-1))^2, C_0(0,0) = 1, psi = prolate-spheroidal taper (reading 6),
 *   K[p][ov][ou][ty][tx] = C_p[ty*beta - off_v][tx*beta - off_u], complex64, each S_p x S_p
 *   matrix contiguous (layout C-1 :1100-1108), plus zeta sums (eq 4.3) kept on the device.
 *   support_table  host [n_wplanes], odd, 1..max_support. NULL = automatic (:1062,:1114, reading 7): per plane
 *                  r = largest |q| on either axis through the centre with |C_p| > 1e-3 (C_0 peak = 1) among
 *                  |q| <= beta*(max_support-1)/2, S_p = 2*ceil(r/beta)+1; bank_dev must then hold
 *                  ig_bank_bytes(ctx, NULL); the call synchronises; read the result with ig_get_supports.
 * Uses work_dev as scratch. Asynchronous. */
ig_status ig_build_wkernels(ig_ctx* ctx, double w_max_lambda, const int* support_table);

/* The support table in use (host int[n_wplanes]). */
ig_status ig_get_supports(ig_ctx* ctx, int* support_table);

/* Test hook: install a bank computed elsewhere (the oracle's), same layout, complex64
 * as float pairs, host memory; zeta sums are recomputed from it. Sets w_max too. */
ig_status ig_debug_set_wkernels(ig_ctx* ctx, double w_max_lambda, const int* support_table,
                                const float* bank_host, size_t bank_bytes);
/* Test hook: copy the device bank to host (complex64 pairs). Synchronises. */
ig_status ig_debug_get_wkernels(ig_ctx* ctx, float* bank_host, size_t bank_bytes);

/* Grid one batch of visibilities, ADDING into the bound grid (eq 4.4). May be called
 * many times (the thesis feeds chunks, :1011). Steps, all on the device:
 *   A2 order rows by baseline (stable, so time stays ascending), records then run
 *      baseline -> channel -> time;  A1 per record: conj flip for w<0 (eq 4.10), nearest
 *      oversampled sample, cell, sub-cell offsets, w-plane (readings 2-4), weighted
 *      visibility (eq 4.16);  A3 records whose footprint leaves the grid or whose weights
 *      are all zero are dropped (:1278,:1315), the stream is cut into work items;
 *   C  the gridder.
 *   uvw_m        dev f64 [nrow][3], metres; a row with a NaN or infinite coordinate is dropped (reading 20)
 *   baseline_id  dev i32 [nrow], any non-negative ids; rows in any order
 *   freqs_hz     HOST f64 [nchan]
 *   vis          dev f32 [nrow][nchan][n_pol][2]
 *   weights      dev f32 [nrow][nchan][n_pol]; weight 0 = flagged (:1286)
 * All arrays dense (no strides) and naturally aligned; with n_pol = 4 vis and weights are read as 16-byte
 * vectors and must be 16-byte aligned (IG_EINVAL otherwise).
 * Asynchronous; inputs must stay valid until the stream reaches the end of the call. */
ig_status ig_grid(ig_ctx* ctx, const double* uvw_m, const int* baseline_id, long long nrow,
                  const double* freqs_hz, int nchan, const float* vis, const float* weights);

/* Same, with HOST inputs: copies them to staging areas inside work_dev and grids. The end-to-end leg.
 * work_dev must hold ig_workspace_bytes(ctx, nrow, nchan) + ig_host_staging_bytes(ctx, nrow, nchan) (an upper
 * bound: a sliced batch needs the workspace of one slice plus two slice-sized staging areas, which is what
 * ig_host_staging_bytes counts for the ig_set_host_slices value in force when it is called). */
size_t ig_host_staging_bytes(const ig_ctx* ctx, long long nrow, int nchan);
/* ig_grid_host cuts the rows into n slices (default 8; 1 = no slicing; batches under 65 536 rows are never
 * sliced) and copies slice k+1 on a second stream while slice k is gridded. The copies overlap the kernels only
 * when the host buffers are pinned. More slices shorten the tracks inside a slice (more commits). */
ig_status ig_set_host_slices(ig_ctx* ctx, int n);
ig_status ig_grid_host(ig_ctx* ctx, const double* uvw_m, const int* baseline_id, long long nrow,
                       const double* freqs_hz, int nchan, const float* vis, const float* weights);

/* ig_grid for a caller that cannot allocate device memory. ig_grid needs a work_dev sized per batch, which
 * somebody must cudaMalloc. A gridding stage that runs inside someone else's process (a correlator pipeline, a
 * framework that has reserved all of HBM for its own pool and hands out fixed input and output buffers), or
 * inside a latency-bound loop where cudaMalloc / cudaFree would stall the whole device, has nobody to ask.
 * This call is ig_grid with its scratch in an array that is part of the library itself (a file-scope
 * __device__ array in csrc/ig_static.cu): same arguments (eq 4.4, steps A1-A3 and C as above), same result up to
 * fp32 summation order; it makes no cudaMalloc / cudaFree call and calls no library routine that allocates device memory.
 *   - Limit: ig_workspace_bytes(ctx, nrow, nchan) <= IG_STATIC_WORK_BYTES (32 MiB; e.g. ~230 000 four-polarisation
 *     records on a 2048^2 grid). A larger batch returns IG_ENOMEM, text in ig_last_error, nothing enqueued: feed
 *     smaller batches (ig_grid* calls add up) or use ig_grid.
 *   - Cost: each GPU this call runs on holds those 32 MiB from the first call until the process exits.
 *   - First call on a GPU: looks up where the array sits on that GPU (once per device, cached; the context's device
 *     must be current, IG_EINVAL if the bound grid lives elsewhere). Make that first call during set-up, before
 *     any stream capture is begun.
 *   - The array is shared by EVERY call on that GPU, whatever the context, and keeps the last call's bytes. The call
 *     clears what it counts in, so calls on one stream may follow each other freely; two calls that can run at the
 *     same time on the GPU (different streams, different host threads' contexts) overwrite each other's
 *     scratch and give wrong grids - order them with events, or give all but one a work buffer and ig_grid.
 *   - ig_bind still asks for a work_dev (the bank builder and the finaliser use it); this call never touches it.
 * The bound work buffer, the statistics, the timing ring and ig_last_launches behave as after ig_grid. */
#define IG_STATIC_WORK_BYTES (32u << 20)
ig_status ig_grid_static(ig_ctx* ctx, const double* uvw_m, const int* baseline_id, long long nrow,
                         const double* freqs_hz, int nchan, const float* vis, const float* weights);

/* Algorithm 4.6: inverse FFT per polarisation (uv origin at pixel (N/2,N/2), +j sign,
 * unnormalised, eq 2.8 :516), real part divided by the normaliser (eq 4.5), the taper
 * (eq 2.9) and the sinc of the nearest-sample lookup (eq 2.13). By default the images are the polarisations
 * themselves; ig_set_stokes_output switches step 2's Stokes conversion on.
 *   image_dev        dev f32 [n_pol][N][N], pixel (N/2,N/2) = phase centre
 *   normaliser_host  HOST f64 [n_pol], receives N_p; may be NULL
 * Uses work_dev (ig_finalize_workspace_bytes()). Synchronises. */
ig_status ig_finalize(ig_ctx* ctx, float* image_dev, double* normaliser_host);

/* Step 2 of Algorithm 4.6, "convert to multiple-Stokes image and normalise". The paper prints no
 * formulas; reading 21: the polarisations are the linear-feed correlations in MeasurementSet order (XX, XY, YX, YY)
 * and, with D_p = image_p / N_p,  I = (D_XX + D_YY)/2, Q = (D_XX - D_YY)/2, U = (D_XY + D_YX)/2, V = (D_XY - D_YX)/(2j)
 * (n_pol = 2 is (XX, YY) -> I, Q; n_pol = 1 -> I = D_0: "only the stokes that can be calculated", :1660).
 * With the switch on, ig_finalize / ig_finalize_channel write image_dev[s] = Stokes parameter s (I, Q, U, V order). */
ig_status ig_set_stokes_output(ig_ctx* ctx, int on);

/* Step C runs two work distributions: records with support < s keep Romein's moving window
 * (registers follow a track, atomics when a pixel leaves the window, :710-742); records with support >= s go to
 * the fixed-tile gather gridder (a warp owns an 8 x 16 pixel tile in registers, records binned by tile, no atomics
 * in the loop). Default 25 (measured crossover on configurations 3-5). s = 1: everything through the gather gridder; s > IG_MAX_SUPPORT: nothing. Same grid
 * up to fp32 summation order. */
ig_status ig_set_gather_min_support(ig_ctx* ctx, int s);

/* Ordering (A2): rows are sorted by (uv tile in Morton order, baseline, time). shift = log2 of the tile side in
 * cells, 5..15; 0 = automatic (N/8 cells, at least 128). A tuning knob for experiments; the grid does not depend on it. */
ig_status ig_set_sort_tile_shift(ig_ctx* ctx, int shift);

/* One grid per channel (the thesis's default mode, :1011, :1120; reading 16): with the switch on, grid_dev holds nchan
 * grids back to back (each ig_grid_bytes(), same layout), channel c of every ig_grid call goes to grid c with its own
 * normaliser, and ig_finalize_channel images one of them. Up to 4096 channels. Switch it before the first ig_grid.
 * Both work distributions serve this mode (the gather gridder's tile plan then covers nchan grids: its bins are
 * (w-plane bucket, channel, tile), 12 B of workspace each, nchan * 16 * (N/32)^2 of them). */
ig_status ig_set_per_channel_grids(ig_ctx* ctx, int on);
ig_status ig_finalize_channel(ig_ctx* ctx, int channel, float* image_dev, double* normaliser_host);

/* eq 4.17: records gridded, records dropped, grid-point updates = sum S^2 * n_pol.
 * Cumulative over ig_grid calls. Synchronises. Any pointer may be NULL. */
ig_status ig_get_stats(ig_ctx* ctx, long long* n_gridded, long long* n_dropped, long long* n_updates);
/* Compression (eq 4.9 :1407-1414): consecutive records of a work item with the same cell,
 * w-plane and sub-cell offsets are summed before gridding. On by default; the grid is the same up to rounding.
 * eq 4.17's update count keeps counting every gridded record (the thesis's "total" rate, :1767).
 * ig_get_compressed: records merged into their predecessor so far. */
ig_status ig_set_compression(ig_ctx* ctx, int on);
ig_status ig_get_compressed(ig_ctx* ctx, long long* n_compressed);
/* Pixel commits so far: atomic reductions of one multi-polarised pixel into the grid (the
 * gridder's red.global.add traffic, for the roofline's byte count). Synchronises. */
ig_status ig_get_commits(ig_ctx* ctx, long long* n_commits);
/* Counting costs a few instructions per grid point and record, so it is off by default: switch it on for
 * the ig_grid calls whose commits are to be counted (bench.py's counted pass). */
ig_status ig_set_commit_counting(ig_ctx* ctx, int on);
/* Measured FP32 FMA peak of the device in TFLOP/s (register-only FFMA loop on every SM, timed
 * with CUDA events on `cuda_stream`): the ALU denominator of the gridding roofline.
 * sink_dev: dev, 4 bytes owned by the caller (written only by a branch that is never taken). */
ig_status ig_measure_fp32_peak(void* cuda_stream, void* sink_dev, double* tflops);
/* Measured rate of the gridder's commit (one 32-byte 4-pol pixel = 2 x red.global.add.v4.f32) at
 * pseudo-random places of buf_dev (dev, `bytes` long, contents are added to), in 1e9 pixel commits/s.
 * |run_len| = consecutive pixels committed by neighbouring lanes (1..32). The SIGN of run_len picks the pixel layout:
 * run_len > 0: the two 16-byte halves of a pixel are neighbours (pixel-interleaved, 32 B per pixel); run_len < 0: the
 * gridder's own 4-pol layout, two planes of polarisation pairs (ig_grid_bytes above), which is the ceiling that
 * applies to ig_grid (bench.py passes -8). 0 or |run_len| > 32: IG_EINVAL. The atomic ceiling of the
 * roofline: L2-resident when bytes << 126 MB, HBM-backed when bytes >> 126 MB. */
ig_status ig_measure_commit_rate(void* cuda_stream, void* buf_dev, size_t bytes, int run_len,
                                 double* gcommits_per_s);
/* Device time split of an ig_grid call in milliseconds (CUDA events recorded on the bound
 * stream): ingest (A1-A3) and gridder (C). calls_back = 0 is the last non-empty call, 1 the one
 * before, ... up to 63. Waits for that call to finish. */
ig_status ig_get_timing(ig_ctx* ctx, int calls_back, float* ingest_ms, float* gridder_ms);
/* The gridder time of that call split into its two work distributions: the moving-window kernel and the
 * fixed-tile gather phase (plan + scatter + gather kernel; 0 when no support reaches ig_set_gather_min_support). */
ig_status ig_get_gridder_split(ig_ctx* ctx, int calls_back, float* window_ms, float* gather_ms);
/* Zero the normaliser and the statistics (for a caller that zeroes the grid to start a new
 * image with the same bank). Asynchronous. */
ig_status ig_reset_accumulators(ig_ctx* ctx);
/* Number of kernels the LAST ig_grid call launched. */
int ig_last_launches(const ig_ctx* ctx);

/* Test hook: the index tuple of every record in INPUT order, six dev i32 arrays
 * [nrow][nchan]: X, Y, off_u, off_v, plane, flags (bit0 = conjugated, bit1 = on grid).
 * Same arithmetic as ig_grid's A1 step. Synchronises. */
ig_status ig_debug_indices(ig_ctx* ctx, const double* uvw_m, long long nrow, const double* freqs_hz,
                           int nchan, int* X, int* Y, int* off_u, int* off_v, int* plane, int* flags);
/* Test hook: the taper psi(eta) the bank builder and the finaliser use, host to host. */
ig_status ig_debug_taper(const double* eta_host, int n, double* psi_host);

#ifdef __cplusplus
}
#endif
#endif /* IG_H */
