// ig_sort.cu - step A2 (ordering): stable LSD radix sort of rows by baseline id.
//
// The thesis groups records by baseline with time ascending on the CPU (Alg 4.5,
// PAPER.md:1613-1646) because the gridder accumulates along a baseline's track (:714).
// Here the rows (nrow <= a few 1e7; records = rows x channels are never moved by the
// sort) are ordered on the device by the 48-bit key (uv tile in Morton order, baseline id):
// 6 passes of an 8-bit stable counting sort, each = per-tile histogram -> exclusive scan
// -> stable scatter. Stability keeps the input (time) order inside a (tile, baseline) run.
// The tile part is new: rows whose footprints fall in the same 2-D region of the grid are
// made neighbours in the work queue, so that the pixel commits of concurrently running
// warps meet in the L2 instead of each costing an HBM read and write-back (round 1's first gridder, without
// the tile key: 1.0 TB of DRAM traffic on config 5 for 24 M touched pixels). A track
// that crosses a tile edge is cut there, which costs one flush of the lane registers.
// Output: perm[j] = input row at sorted place j.
#include "ig_internal.h"

#define SORT_THREADS 256
#define SORT_WARPS (SORT_THREADS / 32)
#define SORT_STEPS 32
#define SORT_TILE (SORT_THREADS * SORT_STEPS)   // 8192 keys per CTA

__device__ __forceinline__ uint32_t lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// per-warp digit counts of this CTA's tile into smem cnt[warp][256]
__device__ __forceinline__ void tile_count(const uint64_t* __restrict__ keys, long long n, int shift,
                                           uint32_t (*cnt)[256]) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&cnt[0][0])[i] = 0;
    __syncthreads();
    const long long base = (long long)blockIdx.x * SORT_TILE + (long long)warp * (32 * SORT_STEPS);
#pragma unroll 4
    for (int s = 0; s < SORT_STEPS; ++s) {
        long long k = base + s * 32 + lane;
        if (k < n) atomicAdd(&cnt[warp][(uint32_t)(keys[k] >> shift) & 255u], 1u);
    }
    __syncthreads();
}

__global__ void __launch_bounds__(SORT_THREADS)
k_sort_hist(const uint64_t* __restrict__ keys, long long n, int shift, uint32_t* __restrict__ hist, int nblk) {
    __shared__ uint32_t cnt[SORT_WARPS][256];
    tile_count(keys, n, shift, cnt);
    uint32_t t = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) t += cnt[w][threadIdx.x];
    hist[(size_t)threadIdx.x * nblk + blockIdx.x] = t;   // bin-major: rows are scanned per bin, bin totals give the bin starts
}

// in-place exclusive scan of rows of m uint32 values, one CTA (any multiple of 32 threads) per row;
// the row total goes to totals[row] when totals != nullptr
__global__ void __launch_bounds__(1024) k_scan_excl(uint32_t* __restrict__ a_all, long long m, uint32_t* __restrict__ totals) {
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t carry_s;
    uint32_t* a = a_all + (size_t)blockIdx.x * m;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (long long t0 = 0; t0 < m; t0 += 4 * blockDim.x) {
        long long i = t0 + (long long)threadIdx.x * 4;
        uint32_t v[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) v[k] = (i + k < m) ? a[i + k] : 0u;
        uint32_t s = v[0] + v[1] + v[2] + v[3], inc = s;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            uint32_t w = lane < nwarp ? wsum[lane] : 0u, wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t y = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += y;
            }
            wsum[lane] = wi - w;   // exclusive over warps; wsum[nwarp..] hold the tile total
        }
        __syncthreads();
        uint32_t carry = carry_s;
        uint32_t ex = carry + wsum[warp] + (inc - s);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (i + k < m) a[i + k] = ex;
            ex += v[k];
        }
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry_s = carry + wsum[warp] + inc;
        __syncthreads();
    }
    if (totals && threadIdx.x == 0) totals[blockIdx.x] = carry_s;
}

// vals_in == nullptr means the identity permutation (first pass)
__global__ void __launch_bounds__(SORT_THREADS)
k_sort_scatter(const uint64_t* __restrict__ keys, const uint32_t* __restrict__ vals_in, long long n, int shift,
               const uint32_t* __restrict__ hist, const uint32_t* __restrict__ binbase, int nblk,
               uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out) {
    __shared__ uint32_t cnt[SORT_WARPS][256];
    tile_count(keys, n, shift, cnt);
    {   // turn per-warp counts into per-warp start positions in the output
        uint32_t run = binbase[threadIdx.x] + hist[(size_t)threadIdx.x * nblk + blockIdx.x];
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            uint32_t c = cnt[w][threadIdx.x];
            cnt[w][threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long base = (long long)blockIdx.x * SORT_TILE + (long long)warp * (32 * SORT_STEPS);
    for (int s = 0; s < SORT_STEPS; ++s) {
        long long k = base + s * 32 + lane;
        bool act = k < n;
        uint64_t key = act ? keys[k] : 0ull;
        uint32_t d = act ? ((uint32_t)(key >> shift) & 255u) : 256u;
        uint32_t peers = __match_any_sync(0xffffffffu, d);
        uint32_t b = act ? cnt[warp][d] : 0u;
        __syncwarp();
        if (act && (peers & lanemask_lt()) == 0) cnt[warp][d] = b + __popc(peers);
        __syncwarp();
        if (act) {
            uint32_t pos = b + __popc(peers & lanemask_lt());
            keys_out[pos] = key;
            vals_out[pos] = vals_in ? vals_in[k] : (uint32_t)k;
        }
    }
}

// key = Morton(tile of the row's grid position at the reference frequency) << 32 | baseline id.
// The position is the one the gridder uses (after the w<0 flip), in cells; it only steers the order.
__device__ __forceinline__ uint32_t spread8(uint32_t x) {
    x &= 0xffu;
    x = (x | (x << 4)) & 0x0f0fu;
    x = (x | (x << 2)) & 0x3333u;
    x = (x | (x << 1)) & 0x5555u;
    return x;
}
__device__ __forceinline__ uint64_t row_key(const double* __restrict__ uvw, const int* __restrict__ baseline_id, long long r,
                                           double cells_per_m, int N, int tile_shift) {
    double u = uvw[3 * r], v = uvw[3 * r + 1], w = uvw[3 * r + 2];
    if (w < 0.0) { u = -u; v = -v; }
    double fx = u * cells_per_m + 0.5 * N, fy = v * cells_per_m + 0.5 * N;
    int x = (int)fmin(fmax(fx, 0.0), (double)(N - 1)), y = (int)fmin(fmax(fy, 0.0), (double)(N - 1));
    uint32_t m = spread8((uint32_t)(x >> tile_shift)) | (spread8((uint32_t)(y >> tile_shift)) << 1);
    return ((uint64_t)m << 32) | (uint32_t)baseline_id[r];
}
__global__ void k_sort_keys(const double* __restrict__ uvw, const int* __restrict__ baseline_id, long long n,
                            double cells_per_m, int N, int tile_shift, uint64_t* __restrict__ keys) {
    long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    keys[r] = row_key(uvw, baseline_id, r, cells_per_m, N, tile_shift);
}

// Small batches (n <= SORT_SMALL_MAX rows: a chunk fed by a streaming caller; configuration 1's 1 792
// rows): the 25 launches of the radix sort cost more than the whole gridding (PAPER.md:2008 makes the same remark
// about preparation on the light configuration). One CTA instead: key and input place are packed into one 64-bit
// word, (48-bit key) << 12 | row, which makes every word distinct, so a plain bitonic network in shared memory
// yields exactly the stable order of the radix sort (ties broken by input place) and needs no scratch.
#define SORT_SMALL_MAX 4096
__global__ void __launch_bounds__(1024)
k_sort_small(const double* __restrict__ uvw, const int* __restrict__ baseline_id, int n, double cells_per_m, int N,
             int tile_shift, uint32_t* __restrict__ perm_out) {
    __shared__ uint64_t s[SORT_SMALL_MAX];
    int np2 = 32;
    while (np2 < n) np2 <<= 1;
    for (int i = threadIdx.x; i < np2; i += blockDim.x)
        s[i] = i < n ? ((row_key(uvw, baseline_id, i, cells_per_m, N, tile_shift) << 12) | (uint64_t)i) : ~0ull;
    __syncthreads();
    for (int k = 2; k <= np2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < (np2 >> 1); t += blockDim.x) {
                const int i = 2 * j * (t / j) + (t % j), l = i + j;      // pair t of this stage: places i < l, j apart
                const bool ascending = (i & k) == 0;
                const uint64_t a = s[i], b = s[l];
                if ((a > b) == ascending) { s[i] = b; s[l] = a; }
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < n; i += blockDim.x) perm_out[i] = (uint32_t)(s[i] & (SORT_SMALL_MAX - 1));
}

size_t ig_sort_scratch_bytes(long long nrow) {
    long long nblk = (nrow + SORT_TILE - 1) / SORT_TILE;
    if (nblk < 1) nblk = 1;
    // keysA, keysB (u64), valsB (valsA is the caller's perm_out), hist
    return 2 * ig_align((size_t)nrow * 8) + ig_align((size_t)nrow * 4) + ig_align((size_t)nblk * 256 * 4) + 1024;
}

int ig_launch_sort_rows(ig_ctx* c, const double* uvw, const int* baseline_id, long long nrow, double ref_freq_hz,
                        uint32_t* perm_out, char* scratch, size_t scratch_bytes) {
    if (nrow >= (1ll << 32)) { c->err = "nrow must be < 2^32"; return -1; }
    if (scratch_bytes < ig_sort_scratch_bytes(nrow)) { c->err = "sort scratch too small"; return -1; }
    int nblk = (int)((nrow + SORT_TILE - 1) / SORT_TILE);
    if (nblk < 1) nblk = 1;
    size_t a8 = ig_align((size_t)nrow * 8), a4 = ig_align((size_t)nrow * 4);
    uint64_t* keysA = (uint64_t*)scratch;
    uint64_t* keysB = (uint64_t*)(scratch + a8);
    uint32_t* valsB = (uint32_t*)(scratch + 2 * a8);
    uint32_t* hist = (uint32_t*)(scratch + 2 * a8 + a4);
    uint32_t* binbase = hist + (size_t)nblk * 256;        // 256 bin totals, scanned to bin start offsets
    uint32_t* valsA = perm_out;
    // 8 x 8 tiles (tile = N/8 cells, at least 128): measured best on configs 4 and 5 (tiles of 1/16..1/4 of
    // the grid side are within 1 %), no effect on the small grids; finer tiles cut too many tracks and make
    // concurrently running warps collide on the same pixels
    int tile_shift = 7;
    while ((c->prm.N >> tile_shift) > 8) ++tile_shift;
    if (c->tile_shift) tile_shift = c->tile_shift;      // ig_set_sort_tile_shift
    const double cells_per_m = ref_freq_hz * c->prm.ku / (double)c->prm.beta;
    if (nrow <= SORT_SMALL_MAX) {
        k_sort_small<<<1, 1024, 0, c->stream>>>(uvw, baseline_id, (int)nrow, cells_per_m, c->prm.N, tile_shift, perm_out);
        IG_CUDA_OK(c, cudaGetLastError());
        return 1;
    }
    k_sort_keys<<<(unsigned)((nrow + 255) / 256), 256, 0, c->stream>>>(uvw, baseline_id, nrow, cells_per_m, c->prm.N,
                                                                      tile_shift, keysA);
    int launches = 1;
    for (int pass = 0; pass < 6; ++pass) {     // bytes 0-3 baseline id, bytes 4-5 Morton tile
        const uint64_t* kin = (pass & 1) ? keysB : keysA;
        const uint32_t* vin = pass == 0 ? nullptr : ((pass & 1) ? valsB : valsA);
        uint64_t* kout = (pass & 1) ? keysA : keysB;
        uint32_t* vout = (pass & 1) ? valsA : valsB;
        k_sort_hist<<<nblk, SORT_THREADS, 0, c->stream>>>(kin, nrow, pass * 8, hist, nblk);
        k_scan_excl<<<256, 256, 0, c->stream>>>(hist, (long long)nblk, binbase);      // one CTA per bin row
        k_scan_excl<<<1, 256, 0, c->stream>>>(binbase, 256, nullptr);
        k_sort_scatter<<<nblk, SORT_THREADS, 0, c->stream>>>(kin, vin, nrow, pass * 8, hist, binbase, nblk, kout, vout);
        launches += 4;
    }
    IG_CUDA_OK(c, cudaGetLastError());
    return launches;   // result is in valsA == perm_out after the 6th pass
}
