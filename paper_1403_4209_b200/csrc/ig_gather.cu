// ig_gather.cu - step C for LARGE supports: the fixed-tile ("gather") gridder and its plan (steps A3 + C).
//
//   grid[Y0+ty][X0+tx][pol] += a[pol] * K[p][ov][ou][ty][tx]      (eq 4.4a/b)
//
// Why a second work distribution. Romein's moving window (ig_gridder.cu) keeps a sum in a
// register only while successive records of ONE track overlap; on long baselines with supports of 17..129 cells
// the window moves by many cells per record, 40-45 % of all register sums end in an atomic (oracle/track_commits.py)
// and the L2 atomic unit, not the FP32 pipe, sets the pace (config 5: 26 G pixel commits). Here the ownership is
// turned round: a warp owns a FIXED 8 x 16 pixel tile of the grid in registers (4 pixels per lane, all
// polarisations), and every record whose footprint crosses the tile - of any baseline, time or channel - is
// accumulated into those registers; the tile is written once per work item. No atomics in the loop, contributions
// of different tracks combine on chip, and the per-(record, pixel) work is a compare, an address, one read-only
// load and the FMAs. The price is lanes outside the footprint (efficiency ~ S/(S+7) * S/(S+3)), so supports below
// `gather_min_support` stay with the moving window, where tracks overlap well and the tile would be mostly idle.
// The thesis had two kernels split at S = 31 for a similar reason (:1371-1379); shared memory is not used for the
// sums (fp32 shared atomics are CAS loops, and a read-modify-write per tap is 4x the FP32 pipe time).
//
// Plan (the thesis's scan / compaction / plan steps, Alg 4.2-4.3 :1446-1508, rebuilt for this ownership):
//   k_index            marks large-support records (IG_HDR_GATHER) and counts them per 32 x 32 "origin tile"
//                      (the tile that holds the footprint's first pixel)
//                      and w-plane bucket: bin = bucket * tiles + tile, bucket-major, so that the kernel matrices
//                      in use at any time stay in L2
//   k_gather_plan_a/b/c  multi-CTA exclusive scan of the bin counts (per-block sums, one CTA over the block sums,
//                      per-block scan with carry) -> bin offsets; cuts every bin's list into items of <= IG_GCH records
//   k_gather_scatter   counting-sort scatter of the marked records into bin order (header rewritten relative
//                      to the tile)
//   k_gather           persistent CTAs; an item's records are staged once into shared memory by the TMA bulk-copy
//                      engine; the CTA's warps take the 8 x 16 sub-tiles of the region the item can reach
//                      (32 + Smax - 1 pixels on a side) from a shared counter; per sub-tile a ballot over the
//                      staged headers finds the records that touch it.
#include "ig_internal.h"

#define IG_GT 32          // origin tile side in pixels
#define IG_GT_SHIFT 5
#ifndef IG_GCH
#define IG_GCH 256        // records per gather item
#endif
#ifndef IG_GW
#define IG_GW 8           // warps per gather CTA
#endif
#define IG_GR 4           // pixel row groups per lane: sub-tile = 8 wide x 4*IG_GR tall
#ifndef IG_XP
#define IG_XP 0          // timing experiments only (results are wrong when non-zero)
#endif
#ifndef IG_GPIPE
#define IG_GPIPE 1       // two records in flight per warp
#endif
#ifndef IG_GCTAS_PER_SM
#define IG_GCTAS_PER_SM 3
#endif

__device__ __forceinline__ uint32_t g_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t g_lanemask_lt() {
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// ---------------------------------------------------------------------------------------------------------
// plan: bin_count[nbins] -> bin_off (exclusive scan), bin_cur (= bin_off, the scatter's cursors), items.
// A bin is (w-plane bucket, origin tile), bucket-major: bin = bucket * ntiles + tile. Items therefore run through the
// grid one plane bucket at a time, and the CTAs in flight read the kernel matrices of ~P/16 planes only: the part of
// the bank in use stays in the 126 MB L2 (config 5: 968 MB bank; with tile-only bins the gather kernel missed L2 on
// a third of its kernel reads and pulled 157 GB from DRAM).
// Three steps so that many CTAs scan: (a) per block of 4096 bins the totals, (b) one CTA scans the block totals,
// (c) per block the bins' offsets and items. plan_hdr[0] = number of items, [1] = number of entries.
__device__ __forceinline__ unsigned long long g_bin_cost(uint32_t c) {       // hi 32 bits: entries, lo 32 bits: items
    return ((unsigned long long)c << 32) | (unsigned long long)((c + IG_GCH - 1) / IG_GCH);
}
// block-wide inclusive scan of one value per thread (1024 threads); returns the inclusive sum, total in *total
__device__ __forceinline__ unsigned long long g_block_scan(unsigned long long v, unsigned long long* wsum, unsigned long long* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        unsigned long long y = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += y;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        unsigned long long w = wsum[lane], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            unsigned long long y = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += y;
        }
        wsum[lane] = wi - w;               // exclusive over warps
        if (lane == 31) wsum[32] = wi;     // block total
    }
    __syncthreads();
    const unsigned long long r = inc + wsum[warp];
    if (total) *total = wsum[32];
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(1024) k_gather_plan_a(const uint32_t* __restrict__ bin_count, unsigned long long* __restrict__ block_sum,
                                                        uint32_t nbins) {
    __shared__ unsigned long long wsum[33];
    const uint32_t i = blockIdx.x * 4096u + threadIdx.x * 4;
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) s += g_bin_cost((i + k < nbins) ? bin_count[i + k] : 0u);
    unsigned long long total;
    g_block_scan(s, wsum, &total);
    if (threadIdx.x == 0) block_sum[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) k_gather_plan_b(unsigned long long* __restrict__ block_sum, uint32_t nblocks,
                                                        uint32_t* __restrict__ plan_hdr) {
    __shared__ unsigned long long wsum[33];
    unsigned long long carry = 0;
    for (uint32_t b0 = 0; b0 < nblocks; b0 += 1024) {
        const uint32_t i = b0 + threadIdx.x;
        const unsigned long long v = i < nblocks ? block_sum[i] : 0ull;
        unsigned long long total;
        const unsigned long long inc = g_block_scan(v, wsum, &total);
        if (i < nblocks) block_sum[i] = carry + inc - v;      // exclusive
        carry += total;
    }
    if (threadIdx.x == 0) { plan_hdr[0] = (uint32_t)carry; plan_hdr[1] = (uint32_t)(carry >> 32); }
}

__global__ void __launch_bounds__(1024) k_gather_plan_c(const uint32_t* __restrict__ bin_count, const unsigned long long* __restrict__ block_sum,
                                                        uint32_t* __restrict__ bin_off, uint32_t* __restrict__ bin_cur,
                                                        uint4* __restrict__ items, uint32_t nbins) {
    __shared__ unsigned long long wsum[33];
    const uint32_t i = blockIdx.x * 4096u + threadIdx.x * 4;
    uint32_t c[4];
    unsigned long long s = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        c[k] = (i + k < nbins) ? bin_count[i + k] : 0u;
        s += g_bin_cost(c[k]);
    }
    const unsigned long long inc = g_block_scan(s, wsum, nullptr);
    unsigned long long ex = block_sum[blockIdx.x] + inc - s;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (i + k < nbins) {
            const uint32_t off = (uint32_t)(ex >> 32), ioff = (uint32_t)ex;
            bin_off[i + k] = off;
            bin_cur[i + k] = off;
            for (uint32_t j = 0, left = c[k]; left; ++j) {
                const uint32_t n = left < IG_GCH ? left : IG_GCH;
                items[ioff + j] = make_uint4(i + k, off + j * IG_GCH, n, 0u);
                left -= n;
            }
        }
        ex += g_bin_cost(c[k]);
    }
}

// ---------------------------------------------------------------------------------------------------------
// scatter: one warp per work item of the record stream (IG_CH records); marked records go to their tile's list.
// Entry (16 + 16 * NPOL bytes): header {ox, oy, S, kbase} (footprint origin relative to the origin tile) followed per
// polarisation by {v_re, v_re, -v_im, v_im}: the two operand pairs of the packed complex multiply-accumulate, so that
// the gridder's shared-memory loads deliver them as aligned register pairs with no arithmetic.
template <int NPOL>
__global__ void __launch_bounds__(256) k_gather_scatter(const char* __restrict__ records, const uint32_t* __restrict__ gcount,
                                                        long long n_chunks, uint32_t* __restrict__ tile_cur, int tiles_x,
                                                        uint32_t ntiles, int n_planes, char* __restrict__ entries, int nchan_grids) {
    constexpr int STRIDE = NPOL == 4 ? 48 : 32;
    constexpr int GSTRIDE = 16 + 16 * NPOL;
    const long long chunk = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (chunk >= n_chunks || gcount[chunk] == 0) return;
    for (int g = 0; g < IG_CH / 32; ++g) {
        const char* rec = records + ((size_t)chunk * IG_CH + g * 32 + lane) * STRIDE;
        const uint4 h = *reinterpret_cast<const uint4*>(rec);
        const bool mine = (h.z & IG_HDR_GATHER) && !(h.z & IG_HDR_MERGED);
        const uint32_t gm = __ballot_sync(0xffffffffu, mine);
        if (!gm) continue;
        if (mine) {
            const int X0 = (int)(h.x & 0xffffu), Y0 = (int)(h.x >> 16);
            // per-channel grids (nchan_grids > 0): the channel of this work item selects the grid, tile = channel * tiles + tile
            const uint32_t tl = (uint32_t)((Y0 >> IG_GT_SHIFT) * tiles_x + (X0 >> IG_GT_SHIFT));
            const uint32_t tile = nchan_grids > 0
                ? ig_gather_bin((int)(h.z & IG_HDR_GPLANE), n_planes, ntiles * (uint32_t)nchan_grids, (uint32_t)(chunk % nchan_grids) * ntiles + tl)
                : ig_gather_bin((int)(h.z & IG_HDR_GPLANE), n_planes, ntiles, tl);
            const uint32_t peers = __match_any_sync(gm, tile);
            const int leader = __ffs(peers) - 1;
            uint32_t base = 0;
            if (lane == leader) base = atomicAdd(&tile_cur[tile], (uint32_t)__popc(peers));
            base = __shfl_sync(peers, base, leader);
            char* e = entries + (size_t)(base + __popc(peers & g_lanemask_lt())) * GSTRIDE;
            *reinterpret_cast<uint4*>(e) = make_uint4((uint32_t)(X0 & (IG_GT - 1)), (uint32_t)(Y0 & (IG_GT - 1)), h.w, h.y);
            float v[8];
            const float4 a = *reinterpret_cast<const float4*>(rec + 16);
            v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
            if constexpr (NPOL == 4) {
                const float4 c = *reinterpret_cast<const float4*>(rec + 32);
                v[4] = c.x; v[5] = c.y; v[6] = c.z; v[7] = c.w;
            }
#pragma unroll
            for (int q = 0; q < NPOL; ++q)
                *reinterpret_cast<float4*>(e + 16 + 16 * q) = make_float4(v[2 * q], v[2 * q], -v[2 * q + 1], v[2 * q + 1]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// One record against one sub-tile (8 columns x 16 rows = 4 row groups of 4 rows, one pixel per lane and row group),
// in two steps so that the kernel values of the NEXT record are in flight while the current one is accumulated
// (a warp's loads are otherwise strictly serial: header -> addresses -> values -> FMAs).
//   g_prepare  header {ox, oy, S, kbase} (footprint origin relative to the origin tile, support, first element of the
//              record's S x S matrix) is a shared-memory broadcast; the lane's tap is (ty0 + 4k, tx) and lies in the
//              footprint iff both are in [0, S); the four kernel values are requested with predicated read-only
//              loads (zero outside the footprint).
//   g_apply    the footprint's rows reach a contiguous range [KA, KB] of the row groups (warp-uniform);
//              g_groups<KA, KB> is the straight-line code for that range: per row group and polarisation
//                acc += (v_re, v_re) * (k_re, k_im);   acc += (-v_im, v_im) * (k_im, k_re)     (two packed FMAs, FFMA2)
//              Row groups outside the range cost nothing, so the lanes wasted in y are at most 3 rows per record.
struct GHit {
    const char* ep;      // the entry in shared memory
    int S, oy;           // support; footprint's first row relative to the sub-tile
    float2 kv[IG_GR];
};

__device__ __forceinline__ void g_prepare(GHit& H, const char* __restrict__ ep, int sub_x, int sub_y, int lx, int lr,
                                          const float2* __restrict__ bank) {
    const int4 h = *reinterpret_cast<const int4*>(ep);              // warp-wide broadcast
    H.ep = ep;
    H.S = h.z;
    H.oy = h.y - sub_y;
    const int tx = lx - (h.x - sub_x);
    const int ty0 = lr - H.oy;
    const bool col_in = (unsigned)tx < (unsigned)h.z;
    const uint32_t e0 = (uint32_t)h.w + (uint32_t)(ty0 * h.z + tx);  // element index of tap (ty0, tx); wraps harmlessly when unused
#pragma unroll
    for (int k = 0; k < IG_GR; ++k) {
        H.kv[k] = make_float2(0.f, 0.f);
#if IG_XP == 1   /* experiment: no kernel loads */
        if (col_in && (unsigned)(ty0 + 4 * k) < (unsigned)h.z) H.kv[k] = make_float2(__uint_as_float(e0 + 4 * k * h.z), 1.f);
#else
        if (col_in && (unsigned)(ty0 + 4 * k) < (unsigned)h.z) H.kv[k] = __ldg(bank + (e0 + (uint32_t)(4 * k * h.z)));
#endif
    }
}

template <int NPOL, int KA, int KB>
__device__ __forceinline__ void g_groups(float2 (&acc)[IG_GR][NPOL], const GHit& H) {
    float2 vre[NPOL], vim[NPOL];
#pragma unroll
    for (int q = 0; q < NPOL; ++q) {
        const float4 t = *reinterpret_cast<const float4*>(H.ep + 16 + 16 * q);   // {v_re, v_re, -v_im, v_im}
        vre[q] = make_float2(t.x, t.y);
        vim[q] = make_float2(t.z, t.w);
    }
#pragma unroll
    for (int k = KA; k <= KB; ++k) {
        const float2 ks = make_float2(H.kv[k].y, H.kv[k].x);
#if IG_XP == 2   /* experiment: one FMA per kernel value */
        acc[k][0] = __ffma2_rn(vre[0], H.kv[k], acc[k][0]);
        (void)ks; (void)vim;
#else
#pragma unroll
        for (int q = 0; q < NPOL; ++q) {
            acc[k][q] = __ffma2_rn(vre[q], H.kv[k], acc[k][q]);
            acc[k][q] = __ffma2_rn(vim[q], ks, acc[k][q]);
        }
#endif
    }
}

template <int NPOL>
__device__ __forceinline__ void g_apply(float2 (&acc)[IG_GR][NPOL], const GHit& H) {
    const int ka = max(H.oy, 0) >> 2, kb = min(H.oy + H.S - 1, 4 * IG_GR - 1) >> 2;   // the record touches the sub-tile: 0 <= ka <= kb <= 3
    switch (ka * 4 + kb) {
#define IG_GCASE(A, B) case A * 4 + B: g_groups<NPOL, A, B>(acc, H); break;
        IG_GCASE(0, 0) IG_GCASE(0, 1) IG_GCASE(0, 2) IG_GCASE(0, 3) IG_GCASE(1, 1) IG_GCASE(1, 2) IG_GCASE(1, 3)
        IG_GCASE(2, 2) IG_GCASE(2, 3) IG_GCASE(3, 3)
#undef IG_GCASE
        default: break;
    }
}

// Iterator over the records of the staged item that touch a sub-tile: ballots over groups of 32 staged headers.
struct GScan {
    const char* buf;
    int count, g0, sub_x, sub_y, lane, gstride;
    uint32_t m;
    __device__ __forceinline__ void start(const char* b, int n, int sx, int sy, int ln, int gs) {
        buf = b; count = n; sub_x = sx; sub_y = sy; lane = ln; gstride = gs; g0 = -32; m = 0u;
    }
    // next touching record (its entry), or nullptr when the item is exhausted; warp-uniform
    __device__ __forceinline__ const char* next() {
        while (m == 0u) {
            g0 += 32;
            if (g0 >= count) return nullptr;
            bool hit = false;
            if (g0 + lane < count) {
                // footprint [ox, ox+S) x [oy, oy+S) against the sub-tile [sub_x, sub_x+8) x [sub_y, sub_y+16)
                const int4 w = *reinterpret_cast<const int4*>(buf + (g0 + lane) * gstride);
                const int ox = w.x - sub_x, oy = w.y - sub_y;
                hit = ox < 8 && ox + w.z > 0 && oy < 4 * IG_GR && oy + w.z > 0;
            }
            m = __ballot_sync(0xffffffffu, hit);
        }
        const int b = __ffs(m) - 1;
        m &= m - 1;
        return buf + (g0 + b) * gstride;
    }
};

template <int NPOL, bool COUNT, bool PERCH>
__global__ void __launch_bounds__(IG_GW * 32, IG_GCTAS_PER_SM)
k_gather(const char* __restrict__ entries, const uint4* __restrict__ items, const uint32_t* __restrict__ plan_hdr,
         float* __restrict__ grid, const float2* __restrict__ bank, int N, int tiles_x, uint32_t ntiles, unsigned* __restrict__ ticket,
         unsigned long long* __restrict__ commits, uint32_t ntiles_v) {
    constexpr int GSTRIDE = 16 + 16 * NPOL;
    __shared__ __align__(128) char buf[IG_GCH * GSTRIDE];
    __shared__ __align__(8) uint64_t bar;
    __shared__ unsigned s_item, s_sub;
    const int lane = threadIdx.x & 31;
    const int lx = lane & 7, lr = lane >> 3;
    const unsigned n_items = plan_hdr[0];
    const unsigned long long plane_bytes = (unsigned long long)N * N * 16;   // 4 pol: two planes of pol pairs
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(g_smem_u32(&bar)), "r"(1) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    uint32_t phase = 0;
    unsigned n_commit = 0;
    for (;;) {
        __syncthreads();                                   // every warp is done with buf, s_item, s_sub
        if (threadIdx.x == 0) { s_item = atomicAdd(ticket, 1u); s_sub = 0; }
        __syncthreads();
        const unsigned it = s_item;
        if (it >= n_items) break;
        const uint4 item = items[it];                      // {tile, first entry, entries, -}
        const int count = (int)item.z;
        if (threadIdx.x == 0) {
            const uint32_t bytes = (uint32_t)count * GSTRIDE;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic reads of buf before the async write
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(g_smem_u32(&bar)), "r"(bytes) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(g_smem_u32(buf)),
                         "l"(entries + (size_t)item.y * GSTRIDE), "r"(bytes), "r"(g_smem_u32(&bar))
                         : "memory");
        }
        asm volatile(
            "{\n.reg .pred p;\nGW_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra GD_%=;\nbra GW_%=;\nGD_%=:\n}\n" ::"r"(
                g_smem_u32(&bar)),
            "r"(phase)
            : "memory");
        phase ^= 1u;
        // largest support of the item -> the region its footprints can reach from the origin tile
        int smax = 0;
        for (int e = lane; e < count; e += 32) smax = max(smax, *reinterpret_cast<const int*>(buf + e * GSTRIDE + 8));
        smax = __reduce_max_sync(0xffffffffu, smax);
        const int nsx = (IG_GT - 1 + smax + 7) >> 3, nsy = (IG_GT - 1 + smax + 4 * IG_GR - 1) / (4 * IG_GR);
        const unsigned nsub = (unsigned)(nsx * nsy);
        // item.x = plane bucket * ntiles_v + channel * ntiles + origin tile (one grid: ntiles_v = ntiles, channel = 0)
        // PERCH (per-channel grids, back to back in memory): grid ch is reached by a row offset, since in every layout
        // ([N][N][npol]; 4 pol: [2][N][N][2]) a whole grid is N (2N for 4 pol) rows of N pixels at the stride pix is scaled by
        int tile_id, row0 = 0;
        if constexpr (PERCH) {
            const uint32_t tile_v = item.x % ntiles_v, ch = tile_v / ntiles;
            tile_id = (int)(tile_v - ch * ntiles);
            row0 = (int)ch * N * (NPOL == 4 ? 2 : 1);
        } else {
            tile_id = (int)(item.x % ntiles);
        }
        const int tile_y = tile_id / tiles_x, tile_x = tile_id - tile_y * tiles_x;
        for (;;) {
            unsigned st = 0;
            if (lane == 0) st = atomicAdd(&s_sub, 1u);
            st = __shfl_sync(0xffffffffu, st, 0);
            if (st >= nsub) break;
            const int sy = (int)st / nsx, sx = (int)st - sy * nsx;
            const int sub_x = sx * 8, sub_y = sy * (4 * IG_GR);        // sub-tile origin relative to the origin tile
            float2 acc[IG_GR][NPOL];
#pragma unroll
            for (int k = 0; k < IG_GR; ++k)
#pragma unroll
                for (int q = 0; q < NPOL; ++q) acc[k][q] = make_float2(0.f, 0.f);
            GScan scan;
            scan.start(buf, count, sub_x, sub_y, lane, GSTRIDE);
            GHit ha, hb;
            const char* e = scan.next();
#if !IG_GPIPE
            (void)hb;
            while (e) {
                g_prepare(ha, e, sub_x, sub_y, lx, lr, bank);
                g_apply<NPOL>(acc, ha);
                e = scan.next();
            }
#else
            // two records in flight: the next one's kernel values are requested before the current one's FMAs
            if (e) {
                g_prepare(ha, e, sub_x, sub_y, lx, lr, bank);
                for (;;) {
                    e = scan.next();
                    if (!e) { g_apply<NPOL>(acc, ha); break; }
                    g_prepare(hb, e, sub_x, sub_y, lx, lr, bank);
                    g_apply<NPOL>(acc, ha);
                    e = scan.next();
                    if (!e) { g_apply<NPOL>(acc, hb); break; }
                    g_prepare(ha, e, sub_x, sub_y, lx, lr, bank);
                    g_apply<NPOL>(acc, hb);
                }
            }
#endif
            // write the sub-tile: one vector reduction per touched pixel and polarisation pair (other items, and the
            // moving-window gridder, add to the same grid)
            const int x = (tile_x << IG_GT_SHIFT) + sub_x + lx;
#pragma unroll
            for (int k = 0; k < IG_GR; ++k) {
                const int y = (tile_y << IG_GT_SHIFT) + sub_y + 4 * k + lr;
                uint32_t any = 0u;
#pragma unroll
                for (int q = 0; q < NPOL; ++q) any |= __float_as_uint(acc[k][q].x) | __float_as_uint(acc[k][q].y);
                if ((any << 1) != 0u && x < N && y < N) {          // some sum is not +-0
                    const size_t pix = (size_t)(row0 + y) * N + x;
                    float a[2 * NPOL];
#pragma unroll
                    for (int q = 0; q < NPOL; ++q) { a[2 * q] = acc[k][q].x; a[2 * q + 1] = acc[k][q].y; }
                    if constexpr (NPOL == 1) {
                        asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(grid + pix * 2), "f"(a[0]), "f"(a[1]) : "memory");
                    } else {
                        float* gp = grid + pix * 4;
                        asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(gp), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3]) : "memory");
                        if constexpr (NPOL == 4) {
                            float* g2 = reinterpret_cast<float*>(reinterpret_cast<char*>(gp) + plane_bytes);
                            asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(g2), "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7]) : "memory");
                        }
                    }
                    if constexpr (COUNT) ++n_commit;
                }
            }
        }
    }
    if constexpr (COUNT) {
        n_commit = __reduce_add_sync(0xffffffffu, n_commit);
        if (lane == 0 && n_commit) atomicAdd(commits, (unsigned long long)n_commit);
    }
}

// ---------------------------------------------------------------------------------------------------------
size_t ig_gather_tiles(const ig_ctx* c) {
    const size_t t = (size_t)((c->prm.N + IG_GT - 1) / IG_GT);
    return t * t;
}
size_t ig_gather_bins(const ig_ctx* c, int nchan) { return ig_gather_tiles(c) * (c->per_channel ? (size_t)nchan : 1) * IG_GBUCKETS; }
size_t ig_gather_max_items(const ig_ctx* c, long long n_chunks, int nchan) {
    return (size_t)n_chunks * IG_CH / IG_GCH + ig_gather_bins(c, nchan) + 1;
}
size_t ig_gather_plan_scratch_bytes(const ig_ctx* c, int nchan) { return ((ig_gather_bins(c, nchan) + 4095) / 4096) * 8; }

int ig_launch_gather(ig_ctx* c, const char* records, const uint32_t* gcount, long long n_chunks, int nchan, uint32_t* tile_count,
                     uint32_t* tile_off, uint32_t* tile_cur, uint4* items, uint32_t* plan_hdr, char* entries,
                     unsigned long long* plan_scratch) {
    if (n_chunks == 0) return 0;
    cudaStream_t stream = c->stream;
    if (ig_gather_bins(c, nchan) >= (1ull << 32)) { c->err = "gather plan: too many (channel, tile) bins"; return -1; }
    const uint32_t ntiles = (uint32_t)ig_gather_tiles(c), nbins = (uint32_t)ig_gather_bins(c, nchan);
    const int nchan_grids = c->per_channel ? nchan : 0;
    const uint32_t ntiles_v = ntiles * (uint32_t)(c->per_channel ? nchan : 1);
    const int tiles_x = (c->prm.N + IG_GT - 1) / IG_GT;
    const uint32_t nblocks = (nbins + 4095u) / 4096u;
    k_gather_plan_a<<<nblocks, 1024, 0, stream>>>(tile_count, plan_scratch, nbins);
    k_gather_plan_b<<<1, 1024, 0, stream>>>(plan_scratch, nblocks, plan_hdr);
    k_gather_plan_c<<<nblocks, 1024, 0, stream>>>(tile_count, plan_scratch, tile_off, tile_cur, items, nbins);
    const unsigned sblocks = (unsigned)((n_chunks + 7) / 8);
    switch (c->prm.npol) {
        case 1: k_gather_scatter<1><<<sblocks, 256, 0, stream>>>(records, gcount, n_chunks, tile_cur, tiles_x, ntiles, c->prm.P, entries, nchan_grids); break;
        case 2: k_gather_scatter<2><<<sblocks, 256, 0, stream>>>(records, gcount, n_chunks, tile_cur, tiles_x, ntiles, c->prm.P, entries, nchan_grids); break;
        default: k_gather_scatter<4><<<sblocks, 256, 0, stream>>>(records, gcount, n_chunks, tile_cur, tiles_x, ntiles, c->prm.P, entries, nchan_grids); break;
    }
    IG_CUDA_OK(c, cudaMemsetAsync(&c->d_acc->ticket_gather, 0, sizeof(unsigned), stream));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    dim3 g((unsigned)(sms * IG_GCTAS_PER_SM)), b(IG_GW * 32);
#define IG_GLAUNCH2(P, C, G) k_gather<P, C, G><<<g, b, 0, stream>>>(entries, items, plan_hdr, c->grid, c->d_bank, c->prm.N, tiles_x, ntiles, &c->d_acc->ticket_gather, &c->d_acc->commits, ntiles_v)
#define IG_GLAUNCH(P, C) do { if (c->per_channel) IG_GLAUNCH2(P, C, true); else IG_GLAUNCH2(P, C, false); } while (0)
    if ((long long)c->prm.N * (c->prm.npol == 4 ? 2 : 1) * (c->per_channel ? nchan : 1) >= (1ll << 31)) { c->err = "per-channel grids: too many grid rows for the gather gridder"; return -1; }
    if (c->count_commits) {
        switch (c->prm.npol) { case 1: IG_GLAUNCH(1, true); break; case 2: IG_GLAUNCH(2, true); break; default: IG_GLAUNCH(4, true); break; }
    } else {
        switch (c->prm.npol) { case 1: IG_GLAUNCH(1, false); break; case 2: IG_GLAUNCH(2, false); break; default: IG_GLAUNCH(4, false); break; }
    }
#undef IG_GLAUNCH2
#undef IG_GLAUNCH
    IG_CUDA_OK(c, cudaGetLastError());
    return 5;
}
