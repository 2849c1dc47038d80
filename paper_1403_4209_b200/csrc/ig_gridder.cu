// ig_gridder.cu - step C, the gridder (eq 4.4a/b).
//
//   grid[Y-h+ty][X-h+tx][pol] += a[pol] * K[p][ov][ou][ty][tx]      for ty,tx in [0,S)
//
// Work distribution. Romein's idea (Fig 2.1) is kept: a lane owns the
// grid points whose coordinates are congruent to its (i,j) modulo the support S, keeps
// their sums in registers while successive records of a track overlap, and commits a
// point with an atomic only when the footprint has moved off it. What is new for sm_100a:
//  - the unit is ONE WARP, not a thread block: a warp owns 32*R points (R <= 8 per lane),
//    so a 9x9 footprint is one warp with R = 3 and a 129x129 one is 65 passes of R = 8;
//    the small supports that dominate W-projection workloads (and that the thesis's
//    256/1024-thread blocks served badly, :1375,:1986) fill the lanes;
//  - work items are fixed-size chunks of IG_CH records taken from a device-side ticket
//    counter by persistent warps - no plan, no host round trip, no tail of idle CTAs;
//  - a chunk is staged into shared memory by the TMA bulk-copy engine (cp.async.bulk +
//    mbarrier), IG_NSTAGE stages in flight per warp; the record header and visibility are
//    then shared-memory broadcasts;
//  - support changes inside a chunk need no flush logic: a lane's point simply changes;
//  - commits are vector reductions, red.global.add.v4.f32: one 4-pol pixel = 2 instructions,
//    one 32-byte L2 sector.
// Kernel values come straight from the bank with read-only loads: each (record, tap) value
// is used once per record, so the only reuse is across records and that lives in L1/L2.
#include "ig_internal.h"

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "W_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra D_%=;\n"
        "bra W_%=;\n"
        "D_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on the mbarrier
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

template <int NPOL>
__device__ __forceinline__ void commit(float* __restrict__ grid, int pix, float (&a)[2 * NPOL]) {
    float* g = grid + (size_t)pix * (2 * NPOL);
    if constexpr (NPOL == 1) {
        asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(g), "f"(a[0]), "f"(a[1]) : "memory");
    } else {
        asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(g), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3]) : "memory");
        if constexpr (NPOL == 4)
            asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(g + 4), "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7]) : "memory");
    }
}

template <int NPOL>
__global__ void __launch_bounds__(IG_GRID_WARPS * 32, 4)
k_gridder(const char* __restrict__ records, const uint32_t* __restrict__ chunk_smax, unsigned n_chunks,
          float* __restrict__ grid, const float2* __restrict__ bank, int N, unsigned* __restrict__ ticket,
          unsigned long long* __restrict__ commits) {
    constexpr int STRIDE = NPOL == 4 ? 48 : 32;
    constexpr int STAGE_BYTES = IG_STAGE * STRIDE;
    __shared__ __align__(128) char sm_rec[IG_GRID_WARPS][IG_CH * STRIDE];
    __shared__ __align__(8) uint64_t sm_bar[IG_GRID_WARPS][IG_NSTAGE];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    char* my_rec = sm_rec[warp];
    uint64_t* my_bar = sm_bar[warp];
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < IG_NSTAGE; ++s) mbar_init(&my_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncwarp();
    uint32_t phase = 0;
    unsigned n_commit = 0;

    for (;;) {
        unsigned chunk = 0;
        if (lane == 0) chunk = atomicAdd(ticket, 1u);
        chunk = __shfl_sync(0xffffffffu, chunk, 0);
        if (chunk >= n_chunks) break;
        const int smax = (int)chunk_smax[chunk];
        if (smax == 0) continue;                       // every record of the item was dropped
        __syncwarp();                                  // all lanes are done with the previous chunk
        if (lane == 0) {
            const char* src = records + (size_t)chunk * (IG_CH * STRIDE);
#pragma unroll
            for (int s = 0; s < IG_NSTAGE; ++s) {
                mbar_expect_tx(&my_bar[s], STAGE_BYTES);
                tma_load_1d(my_rec + s * STAGE_BYTES, src + s * STAGE_BYTES, STAGE_BYTES, &my_bar[s]);
            }
        }
        const int s2max = smax * smax;
        const int n_pass = (s2max + 32 * IG_RMAX - 1) / (32 * IG_RMAX);
        const int R = (s2max + 32 * n_pass - 1) / (32 * n_pass);   // points per lane, <= IG_RMAX

        for (int pass = 0; pass < n_pass; ++pass) {
            const int q0 = pass * 32 * R + lane;
            float acc[IG_RMAX][2 * NPOL];
            int prev[IG_RMAX];
            uint32_t ij[IG_RMAX];
#pragma unroll
            for (int k = 0; k < IG_RMAX; ++k) {
                prev[k] = -1; ij[k] = 0xffffffffu;
#pragma unroll
                for (int e = 0; e < 2 * NPOL; ++e) acc[k][e] = 0.f;
            }
            int curS = 0;
            for (int st = 0; st < IG_NSTAGE; ++st) {
                if (pass == 0) mbar_wait(&my_bar[st], phase);
                const char* rp = my_rec + st * STAGE_BYTES;
                for (int r = 0; r < IG_STAGE; ++r, rp += STRIDE) {
                    const uint4 h = *reinterpret_cast<const uint4*>(rp);
                    const int S = (int)((h.z >> 16) & 0xffu);
                    if (S == 0) continue;              // dropped record (step A3)
                    if (S != curS) {                   // new support: re-derive the owned residues
                        curS = S;
#pragma unroll
                        for (int k = 0; k < IG_RMAX; ++k) {
                            if (k < R) {
                                const int q = q0 + k * 32;
                                const int j = q / S;
                                ij[k] = (q < S * S) ? (uint32_t)((q - j * S) | (j << 8)) : 0xffffffffu;
                            }
                        }
                    }
                    const int cm = (int)(h.z & 0xffu), dm = (int)((h.z >> 8) & 0xffu);
                    float v[2 * NPOL];
                    {
                        const float4 a = *reinterpret_cast<const float4*>(rp + 16);
                        v[0] = a.x; v[1] = a.y;
                        if constexpr (NPOL >= 2) { v[2] = a.z; v[3] = a.w; }
                        if constexpr (NPOL == 4) {
                            const float4 b = *reinterpret_cast<const float4*>(rp + 32);
                            v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
                        }
                    }
                    const float2* kb = bank + h.y;
                    float2 kv[IG_RMAX];
                    int pix[IG_RMAX];
#pragma unroll
                    for (int k = 0; k < IG_RMAX; ++k) {
                        if (k < R && ij[k] != 0xffffffffu) {
                            int tx = (int)(ij[k] & 0xffu) + cm; tx = tx >= S ? tx - S : tx;
                            int ty = (int)(ij[k] >> 8) + dm;    ty = ty >= S ? ty - S : ty;
                            pix[k] = (int)h.x + ty * N + tx;
                            kv[k] = __ldg(kb + ty * S + tx);
                        }
                    }
#pragma unroll
                    for (int k = 0; k < IG_RMAX; ++k) {
                        if (k < R && ij[k] != 0xffffffffu) {
                            if (pix[k] != prev[k]) {
                                if (prev[k] >= 0) { commit<NPOL>(grid, prev[k], acc[k]); ++n_commit; }
#pragma unroll
                                for (int e = 0; e < 2 * NPOL; ++e) acc[k][e] = 0.f;
                                prev[k] = pix[k];
                            }
#pragma unroll
                            for (int q = 0; q < NPOL; ++q) {
                                acc[k][2 * q] = fmaf(v[2 * q], kv[k].x, acc[k][2 * q]);
                                acc[k][2 * q] = fmaf(-v[2 * q + 1], kv[k].y, acc[k][2 * q]);
                                acc[k][2 * q + 1] = fmaf(v[2 * q], kv[k].y, acc[k][2 * q + 1]);
                                acc[k][2 * q + 1] = fmaf(v[2 * q + 1], kv[k].x, acc[k][2 * q + 1]);
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < IG_RMAX; ++k)
                if (k < R && prev[k] >= 0) { commit<NPOL>(grid, prev[k], acc[k]); ++n_commit; }
        }
        phase ^= 1u;
    }
    n_commit = __reduce_add_sync(0xffffffffu, n_commit);
    if (lane == 0 && n_commit) atomicAdd(commits, (unsigned long long)n_commit);
}

int ig_launch_gridder(ig_ctx* c, const char* records, const uint32_t* chunk_smax, long long n_chunks) {
    if (n_chunks == 0) return 0;
    if (n_chunks >= (1ll << 32) - 65536) { c->err = "too many work items"; return -1; }
    IG_CUDA_OK(c, cudaMemsetAsync(&c->d_acc->ticket, 0, sizeof(unsigned), c->stream));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int per_sm = 4;
    long long want = (n_chunks + IG_GRID_WARPS - 1) / IG_GRID_WARPS;
    unsigned ctas = (unsigned)(want < (long long)sms * per_sm ? want : (long long)sms * per_sm);
    dim3 g(ctas), b(IG_GRID_WARPS * 32);
    switch (c->prm.npol) {
        case 1: k_gridder<1><<<g, b, 0, c->stream>>>(records, chunk_smax, (unsigned)n_chunks, c->grid, c->d_bank, c->prm.N, &c->d_acc->ticket, &c->d_acc->commits); break;
        case 2: k_gridder<2><<<g, b, 0, c->stream>>>(records, chunk_smax, (unsigned)n_chunks, c->grid, c->d_bank, c->prm.N, &c->d_acc->ticket, &c->d_acc->commits); break;
        default: k_gridder<4><<<g, b, 0, c->stream>>>(records, chunk_smax, (unsigned)n_chunks, c->grid, c->d_bank, c->prm.N, &c->d_acc->ticket, &c->d_acc->commits); break;
    }
    IG_CUDA_OK(c, cudaGetLastError());
    return 1;
}
