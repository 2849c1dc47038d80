// ig_internal.h - shared declarations of the CUDA path (never included by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/ig.h"

#define IG_CH 128            // records per chunk (one work item per (row block, channel))
#define IG_STAGE 32          // records per TMA stage
#define IG_NSTAGE (IG_CH / IG_STAGE)
#ifndef IG_RMAX
#define IG_RMAX 4
#endif
// IG_RMAX: grid points per lane, at most (tunable with -DIG_RMAX for experiments)
#define IG_TIMING_RING 64    // ig_grid calls whose event triples are kept
#ifndef IG_GRID_CTAS_PER_SM
#define IG_GRID_CTAS_PER_SM 5
#endif
// IG_GRID_CTAS_PER_SM: launch bound and persistent grid size
// Record header word z (16-byte header {pix_base, kbase, z, plane}): Romein offsets c, d (eq 4.7) and the
// support S in 9 bits each (S <= 511, the largest support the thesis sweeps), then flags.
#define IG_HDR_C(z) ((int)((z) & 0x1ffu))
#define IG_HDR_D(z) ((int)(((z) >> 9) & 0x1ffu))
#define IG_HDR_S(z) ((int)(((z) >> 18) & 0x1ffu))
#define IG_HDR_PACK(c, d, S) ((uint32_t)(c) | ((uint32_t)(d) << 9) | ((uint32_t)(S) << 18))
#define IG_HDR_WINDOW 0x07ffffffu  // c, d, S: with pix_base, the window a record's footprint occupies
#define IG_HDR_CONJ (1u << 27)     // visibility was conjugated (w < 0, eq 4.10)
#define IG_HDR_MERGED (1u << 28)   // visibility already summed into the run's head record (compression)
// Large-support record that the fixed-tile gather gridder handles (ig_gather.cu). Its header is
// {X0 | Y0 << 16, kbase, flags (c = d = S = 0, so the moving-window gridder sees a skip record), S}.
#define IG_HDR_GATHER (1u << 29)
#define IG_HDR_GPLANE 0x0003ffffu   // gather records: the w-plane (clamped to 18 bits; only a locality hint for the plan) in the c, d bits of word z, S stays 0
#define IG_GBUCKETS 16             // w-plane buckets of the gather plan: bin = bucket * tiles + origin tile
#define IG_GATHER_MIN_DEFAULT 25   // supports >= this go to the gather gridder (ig_set_gather_min_support)
#define IG_MAX_CHAN_GRIDS 4096   // per-channel grid mode: channels whose normalisers the bank head has room for
#define IG_GRID_WARPS 4      // warps per gridder CTA

// Device-side tail of the bank buffer: small tables and accumulators.
struct IgPlaneEntry { int support; uint32_t koff; uint32_t magic; uint32_t pad_; };   // koff in complex elements; magic = floor(2^32/S)+1: x/S == umulhi(x, magic) for x < 2^23 (S = 1: 2^32-1, see install_table)
struct IgAccum {
    double norm[4];                     // eq 4.5 normaliser per polarisation
    unsigned long long gridded, dropped, updates;   // eq 4.17
    unsigned long long merged;          // records pre-summed into their predecessor (compression)
    unsigned long long commits;         // pixel commits (atomic reductions of one multi-pol pixel) by the gridder
    unsigned int ticket;                // work queue of the moving-window gridder
    unsigned int ticket_gather;         // work queue of the gather gridder
};

struct IgParams {            // passed by value to kernels
    int N, beta, P, npol;
    int shift;               // ceil(beta/2) - 1
    int bshift;              // log2(beta) when beta is a power of two, else -1
    double ku, kw;           // index constants (include/ig.h, DESIGN.md C.1)
};

struct ig_ctx {
    IgParams prm{};
    double cell_rad = 0, du = 0, w_max = 0;
    int max_support = 0;
    // bound buffers
    float* grid = nullptr; size_t grid_bytes = 0;
    char* work = nullptr; size_t work_bytes = 0;
    char* bank_buf = nullptr; size_t bank_bytes = 0;
    cudaStream_t stream = nullptr;
    bool bound = false, have_bank = false;
    int host_slices = 8;                      // ig_set_host_slices
    cudaStream_t copy_stream = nullptr;       // ig_grid_host: H2D copies of the next slice
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_free[2] = {nullptr, nullptr};
    bool per_channel = false;                 // ig_set_per_channel_grids: one grid per channel (thesis default, :1120)
    double* d_chan_norm = nullptr;            // [IG_MAX_CHAN_GRIDS][4] normalisers of the per-channel grids
    bool compress = true;                     // ig_set_compression
    int tile_shift = 0;                       // ig_set_sort_tile_shift (0 = automatic: N/8 cells, at least 128)
    int gather_min = IG_GATHER_MIN_DEFAULT;   // ig_set_gather_min_support
    bool count_commits = false;               // ig_set_commit_counting
    bool stokes = false;                      // ig_set_stokes_output: the finaliser writes I,Q,U,V instead of the correlations
    // bank description (host copies)
    std::vector<int> support;
    std::vector<uint32_t> koff;
    size_t bank_elems = 0;
    // device pointers inside bank_buf
    float2* d_bank = nullptr; double* d_zeta = nullptr; IgPlaneEntry* d_planes = nullptr;
    IgAccum* d_acc = nullptr;
    // timing of the last ig_grid
    cudaEvent_t ev[IG_TIMING_RING][4] = {};   // ring over the last ig_grid calls: start, after ingest, after the moving-window gridder, end
    long long n_timed = 0;                    // ig_grid calls timed so far
    int launches = 0;
    std::string err;
};

// Can any record of an ig_grid call go to the gather gridder? Not when no plane's support reaches the threshold.
// Before a support table is installed the answer is the cautious one. Decides whether the plan arrays and the entry
// area of the workspace exist at all.
static inline bool ig_gather_possible(const ig_ctx* c) {
    if (c->support.empty()) return c->max_support >= c->gather_min;
    for (int s : c->support) if (s >= c->gather_min) return true;
    return false;
}
static inline size_t ig_align(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }
static inline int ig_rec_stride(int npol) { return npol == 4 ? 48 : 32; }  // bytes, multiple of 16

// the taper psi(eta), host code in ig_bank.cu
void ig_taper_eval(const double* eta, int n, double* psi);

// launchers (each returns the number of kernels launched, or -1 with ctx->err set)
int ig_launch_sort_rows(ig_ctx* c, const double* uvw, const int* baseline_id, long long nrow, double ref_freq_hz,
                        uint32_t* perm_out, char* scratch, size_t scratch_bytes);
size_t ig_sort_scratch_bytes(long long nrow);
// (compression is applied in k_index when c->compress is set)
int ig_launch_index(ig_ctx* c, const double* uvw, const uint32_t* perm, long long nrow,
                    const double* d_freqs, int nchan, const float* vis, const float* wt,
                    char* records, uint32_t* chunk_smax, uint32_t* gcount, uint32_t* tile_count, int gather_min);   // uses c->per_channel / c->d_chan_norm
// gather gridder (ig_gather.cu): plan, scatter, gridder; gcount[chunk] = marked records per work item
// With per-channel grids (c->per_channel) the plan covers nchan grids: the "tile" of a bin is then channel * tiles + tile.
size_t ig_gather_tiles(const ig_ctx* c);
size_t ig_gather_bins(const ig_ctx* c, int nchan);
size_t ig_gather_plan_scratch_bytes(const ig_ctx* c, int nchan);
// plan bin of a gather record (both k_index and k_gather_scatter call it)
__host__ __device__ static inline uint32_t ig_gather_bin(int plane, int n_planes, uint32_t ntiles, uint32_t tile) {
    return (uint32_t)(((long long)plane * IG_GBUCKETS) / n_planes) * ntiles + tile;
}
size_t ig_gather_max_items(const ig_ctx* c, long long n_chunks, int nchan);
int ig_launch_gather(ig_ctx* c, const char* records, const uint32_t* gcount, long long n_chunks, int nchan, uint32_t* tile_count,
                     uint32_t* tile_off, uint32_t* tile_cur, uint4* items, uint32_t* plan_hdr, char* entries,
                     unsigned long long* plan_scratch);
int ig_launch_debug_index(ig_ctx* c, const double* uvw, long long nrow, const double* d_freqs, int nchan,
                          int* X, int* Y, int* ou, int* ov, int* pl, int* fl);
int ig_launch_gridder(ig_ctx* c, const char* records, const uint32_t* chunk_smax, long long nrb, int nchan);
int ig_launch_bank(ig_ctx* c, char* scratch, size_t scratch_bytes);
size_t ig_bank_scratch_bytes(const ig_ctx* c);
int ig_launch_zeta(ig_ctx* c);
int ig_detect_supports(ig_ctx* c, char* scratch, size_t scratch_bytes, int* table);
int ig_run_finalize(ig_ctx* c, int channel, float* image, double* norm_host, bool stokes);   // channel < 0: the single grid
size_t ig_finalize_scratch_bytes(const ig_ctx* c);

#define IG_CUDA_OK(ctx, call)                                                        \
    do {                                                                             \
        cudaError_t e_ = (call);                                                     \
        if (e_ != cudaSuccess) {                                                     \
            (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);         \
            return -1;                                                               \
        }                                                                            \
    } while (0)
