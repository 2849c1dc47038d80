// ig_gridder.cu - step C, the gridder (eq 4.4a/b).
//
//   grid[Y-h+ty][X-h+tx][pol] += a[pol] * K[p][ov][ou][ty][tx]      for ty,tx in [0,S)
//
// Work distribution. Romein's idea (Fig 2.1) is kept: a lane owns the
// grid points whose coordinates are congruent to its (i,j) modulo the support S, keeps
// their sums in registers while successive records of a track overlap, and commits a
// point with an atomic only when the footprint has moved off it. What is new for sm_100a:
//  - the unit is ONE WARP, not a thread block: a warp owns 32*R points (R <= IG_RMAX = 4 per lane),
//    so a 9x9 footprint is one pass with R = 3 and a 129x129 one is 131 passes of R = 4;
//    the small supports that dominate W-projection workloads (and that the thesis's
//    256/1024-thread blocks served badly, :1375,:1986) fill the lanes;
//  - work items are fixed-size chunks of IG_CH records taken from a device-side ticket
//    counter by persistent warps - no plan, no host round trip, no tail of idle CTAs;
//  - a chunk is staged into shared memory by the TMA bulk-copy engine (cp.async.bulk +
//    mbarrier), IG_NSTAGE stages in flight per warp; the record header and visibility are
//    then shared-memory broadcasts;
//  - support changes inside a chunk need no flush logic: a lane's point simply changes;
//  - commits are vector reductions, red.global.add.v4.f32. The 4-pol grid is stored as two planes of
//    polarisation pairs, so a pixel commit is 2 instructions of 16 bytes and NEIGHBOURING lanes (consecutive
//    x) share a 32-byte sector: half the L2 atomic sector operations of a pixel-interleaved layout
//    (measured 174 vs 110 G pixel commits/s, ig_measure_commit_rate).
// Kernel values come straight from the bank with read-only loads: each (record, tap) value
// is used once per record, so the only reuse is across records and that lives in L1/L2.
#include "ig_internal.h"
#ifndef IG_XP
#define IG_XP 0          // timing experiments only (results are wrong when non-zero)
#endif

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

// Packed fp32 pairs (sm_100a FFMA2, PTX fma.rn.f32x2): one complex accumulator = one 64-bit register
// pair (re, im); a complex multiply-accumulate acc += v * k is exactly two FFMA2
//   (re,im) += (v_re, v_re) * (k_re, k_im);   (re,im) += (-v_im, v_im) * (k_im, k_re)
// - ptxas folds the broadcast, the swap and the half negation into operand modifiers (.F32, .LO_HI, .NP).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ void cmac(f32x2& acc, float v_re, float v_im, f32x2 k) {
    float k_re, k_im;
    unpack2(k, k_re, k_im);
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(pack2(v_re, v_re)), "l"(k));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc) : "l"(pack2(-v_im, v_im)), "l"(pack2(k_im, k_re)));
}

// Commit step of one owned point, branch-free: if the record's pixel differs from the one the lane
// holds, the held sums go to the grid with vector reductions (unless the lane held nothing, prev < 0),
// the sums restart from zero and the lane takes the new pixel. Written as predicated PTX so that the
// sums stay in place. COUNT adds the commit counter (ig_get_commits).
template <int NPOL, bool COUNT>
__device__ __forceinline__ void commit_step(f32x2 (&a)[NPOL], int& prev, int pix, float* __restrict__ grid,
                                            unsigned long long plane_bytes, unsigned& n_commit) {
    if constexpr (COUNT) n_commit += (pix != prev && prev >= 0) ? 1u : 0u;
    if constexpr (NPOL == 4) {
        asm volatile(
            "{\n\t.reg .pred p, q;\n\t.reg .u64 ad, ae;\n\t.reg .f32 f<8>;\n\t"
            "setp.ne.s32 p, %5, %4;\n\t"
            "setp.ge.and.s32 q, %4, 0, p;\n\t"
            "mov.b64 {f0,f1}, %0;\n\tmov.b64 {f2,f3}, %1;\n\tmov.b64 {f4,f5}, %2;\n\tmov.b64 {f6,f7}, %3;\n\t"
            "mad.wide.s32 ad, %4, 16, %6;\n\t"
            "add.u64 ae, ad, %7;\n\t"
            "@q red.global.add.v4.f32 [ad], {f0,f1,f2,f3};\n\t"
            "@q red.global.add.v4.f32 [ae], {f4,f5,f6,f7};\n\t"
            "@p mov.b64 %0, 0;\n\t@p mov.b64 %1, 0;\n\t@p mov.b64 %2, 0;\n\t@p mov.b64 %3, 0;\n\t"
            "@p mov.s32 %4, %5;\n\t}"
            : "+l"(a[0]), "+l"(a[1]), "+l"(a[2]), "+l"(a[3]), "+r"(prev)
            : "r"(pix), "l"(grid), "l"(plane_bytes));
    } else if constexpr (NPOL == 2) {
        asm volatile(
            "{\n\t.reg .pred p, q;\n\t.reg .u64 ad;\n\t.reg .f32 f<4>;\n\t"
            "setp.ne.s32 p, %3, %2;\n\t"
            "setp.ge.and.s32 q, %2, 0, p;\n\t"
            "mov.b64 {f0,f1}, %0;\n\tmov.b64 {f2,f3}, %1;\n\t"
            "@q mad.wide.s32 ad, %2, 16, %4;\n\t"
            "@q red.global.add.v4.f32 [ad], {f0,f1,f2,f3};\n\t"
            "@p mov.b64 %0, 0;\n\t@p mov.b64 %1, 0;\n\t"
            "@p mov.s32 %2, %3;\n\t}"
            : "+l"(a[0]), "+l"(a[1]), "+r"(prev)
            : "r"(pix), "l"(grid));
    } else {
        asm volatile(
            "{\n\t.reg .pred p, q;\n\t.reg .u64 ad;\n\t.reg .f32 f<2>;\n\t"
            "setp.ne.s32 p, %2, %1;\n\t"
            "setp.ge.and.s32 q, %1, 0, p;\n\t"
            "mov.b64 {f0,f1}, %0;\n\t"
            "@q mad.wide.s32 ad, %1, 8, %3;\n\t"
            "@q red.global.add.v2.f32 [ad], {f0,f1};\n\t"
            "@p mov.b64 %0, 0;\n\t"
            "@p mov.s32 %1, %2;\n\t}"
            : "+l"(a[0]), "+r"(prev)
            : "r"(pix), "l"(grid));
    }
}

// final flush of one point
template <int NPOL>
__device__ __forceinline__ void commit(float* __restrict__ grid, unsigned long long plane_bytes, int pix, f32x2 (&acc)[NPOL]) {
    float a[2 * NPOL];
#pragma unroll
    for (int q = 0; q < NPOL; ++q) unpack2(acc[q], a[2 * q], a[2 * q + 1]);
    if constexpr (NPOL == 1) {
        float* g = grid + (size_t)pix * 2;
        asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(g), "f"(a[0]), "f"(a[1]) : "memory");
    } else {
        float* g = grid + (size_t)pix * 4;       // one plane holds a polarisation pair per pixel
        asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(g), "f"(a[0]), "f"(a[1]), "f"(a[2]), "f"(a[3]) : "memory");
        if constexpr (NPOL == 4) {
            float* g2 = reinterpret_cast<float*>(reinterpret_cast<char*>(g) + plane_bytes);
            asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(g2), "f"(a[4]), "f"(a[5]), "f"(a[6]), "f"(a[7]) : "memory");
        }
    }
}

// One pass of one warp over a RUN of records of equal support S (contiguous in the staged item):
// the lane owns the R points q = q0 + 32k of the S x S footprint. Control flow is warp-uniform.
// Lanes whose q lies outside the footprint run the same instructions on tap (0,0) with the sentinel
// pixel -1, which never commits.
template <int NPOL, int R, bool COUNT>
__device__ __forceinline__ unsigned grid_run(const char* __restrict__ rp, int n_rec, int S, int q0,
                                             float* __restrict__ grid, const float2* __restrict__ bank, int N) {
    constexpr int STRIDE = NPOL == 4 ? 48 : 32;
    const unsigned long long plane_bytes = (unsigned long long)N * N * 16;   // 4 pol: two planes of pol pairs
    f32x2 acc[R][NPOL];
    int prev[R], ii[R], jj[R];
    uint32_t amask = 0;
#pragma unroll
    for (int k = 0; k < R; ++k) {
        const int q = q0 + k * 32;
        const int j = q / S;
        const bool act = q < S * S;
        ii[k] = act ? q - j * S : 0;
        jj[k] = act ? j : 0;
        amask |= act ? (1u << k) : 0u;
        prev[k] = -1;
#pragma unroll
        for (int e = 0; e < NPOL; ++e) acc[k][e] = 0ull;
    }
    const unsigned long long* __restrict__ bank64 = reinterpret_cast<const unsigned long long*>(bank);
    unsigned n_commit = 0;
    uint32_t krel[R];                  // tap index ty*S+tx of each point for the current window position
#pragma unroll
    for (int k = 0; k < R; ++k) krel[k] = 0;
    uint32_t last_x = 0xffffffffu, last_z = 0xffffffffu;
#pragma unroll 1
    for (int r = 0; r < n_rec; ++r, rp += STRIDE) {
        const uint4 h = *reinterpret_cast<const uint4*>(rp);
        if (h.z & IG_HDR_MERGED) continue;   // compression: ingest summed this record into its predecessor
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
        f32x2 kv[R];
        // Same window as the record before (same cell; only the sub-cell offsets, hence the kernel matrix,
        // may differ): every lane keeps its pixels and taps, so the index arithmetic and the commit test
        // are skipped. Slow baselines stay in a cell for many records (warp-uniform branch).
        const bool same = (h.x == last_x) && ((h.z & IG_HDR_WINDOW) == last_z);
        if (same) {
#pragma unroll
#if IG_XP == 1
            for (int k = 0; k < R; ++k) kv[k] = (unsigned long long)(krel[k] + h.y) | (0x3f800000ull << 32);
#else
            for (int k = 0; k < R; ++k) kv[k] = __ldg(bank64 + (uint32_t)(krel[k] + h.y));
#endif
        } else {
            last_x = h.x; last_z = h.z & IG_HDR_WINDOW;
            const int cm = IG_HDR_C(h.z), dm = IG_HDR_D(h.z);
            int pix[R];
#pragma unroll
            for (int k = 0; k < R; ++k) {
                const int tu = ii[k] + cm, tv = jj[k] + dm;
                const int tx = (int)min((unsigned)tu, (unsigned)(tu - S));     // (i + c) mod S
                const int ty = (int)min((unsigned)tv, (unsigned)(tv - S));
                pix[k] = (amask & (1u << k)) ? ty * N + ((int)h.x + tx) : -1;
                krel[k] = (uint32_t)(ty * S + tx);
#if IG_XP == 1
                kv[k] = (unsigned long long)(krel[k] + h.y) | (0x3f800000ull << 32);
#else
                kv[k] = __ldg(bank64 + (uint32_t)(krel[k] + h.y));            // 32-bit element index
#endif
            }
#pragma unroll
            for (int k = 0; k < R; ++k) {
                // warp-uniform skip: in about half of the (record, slot) pairs no lane's pixel has changed
#if IG_XP == 3   /* experiment: no commits */
                prev[k] = pix[k];
#else
                if (__any_sync(0xffffffffu, pix[k] != prev[k]))
                    commit_step<NPOL, COUNT>(acc[k], prev[k], pix[k], grid, plane_bytes, n_commit);
#endif
            }
        }
#pragma unroll
        for (int k = 0; k < R; ++k) {
#if IG_XP == 2
            cmac(acc[k][0], v[0], v[1], kv[k]);
#else
#pragma unroll
            for (int q = 0; q < NPOL; ++q) cmac(acc[k][q], v[2 * q], v[2 * q + 1], kv[k]);
#endif
        }
    }
#pragma unroll
    for (int k = 0; k < R; ++k)
        if (prev[k] >= 0) { commit<NPOL>(grid, plane_bytes, prev[k], acc[k]); ++n_commit; }
    return n_commit;
}

template <int NPOL, bool COUNT>
__global__ void __launch_bounds__(IG_GRID_WARPS * 32, IG_GRID_CTAS_PER_SM)
k_gridder(const char* __restrict__ records, const uint32_t* __restrict__ chunk_smax, unsigned nrb, unsigned nchan,
          float* __restrict__ grid, const float2* __restrict__ bank, int N, unsigned* __restrict__ ticket,
          unsigned long long* __restrict__ commits, size_t chan_stride, bool two_phase) {
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
    const unsigned n_chunks = nrb * nchan;

    for (;;) {
        unsigned tk = 0;
        if (lane == 0) tk = atomicAdd(ticket, 1u);
        tk = __shfl_sync(0xffffffffu, tk, 0);
        // Small batches (two_phase): the queue is walked twice, first the items with multi-pass supports, then the rest, so
        // that the expensive items are not left for the end (longest-first; matters when a warp gets only tens of items)
        if (tk >= (two_phase ? 2u * n_chunks : n_chunks)) break;
        const bool second = tk >= n_chunks;
        const unsigned ti = second ? tk - n_chunks : tk;
        // tickets run channel-major: neighbours in the queue are neighbouring row blocks of ONE channel
        const unsigned ch = ti / nrb;
        const unsigned chunk = (ti - ch * nrb) * nchan + ch;
        float* __restrict__ grid_ch = grid + (size_t)ch * chan_stride;   // per-channel grids: chan_stride = floats per grid, else 0
        const unsigned sm_item = chunk_smax[chunk];
        if (sm_item == 0) continue;                    // every record of the item was dropped
        if (two_phase && ((sm_item >= 13u) == second)) continue;
        __syncwarp();                                  // all lanes are done with the previous item
        if (lane == 0) {
            const char* src = records + (size_t)chunk * (IG_CH * STRIDE);
#pragma unroll
            for (int s = 0; s < IG_NSTAGE; ++s) {
                mbar_expect_tx(&my_bar[s], STAGE_BYTES);
                tma_load_1d(my_rec + s * STAGE_BYTES, src + s * STAGE_BYTES, STAGE_BYTES, &my_bar[s]);
            }
        }
        // Cut the item into runs of equal support. A support change re-maps every lane's residues, so all
        // points commit there anyway (Romein's scheme flushes on a support change too); per
        // run the pass count and R are then the best fit for that support, not for the item's largest one.
        uint32_t bnd[IG_NSTAGE];                       // bit r of bnd[g]: record 32g+r starts a run
        int s_prev = -1;
#pragma unroll
        for (int g = 0; g < IG_NSTAGE; ++g) {
            mbar_wait(&my_bar[g], phase);
            const int sv = IG_HDR_S(*reinterpret_cast<const uint32_t*>(my_rec + (g * 32 + lane) * STRIDE + 8));
            int before = __shfl_up_sync(0xffffffffu, sv, 1);
            if (lane == 0) before = s_prev;
            bnd[g] = __ballot_sync(0xffffffffu, sv != before);
            s_prev = __shfl_sync(0xffffffffu, sv, 31);
        }
        int r0 = 0;
        while (r0 < IG_CH) {
            // end of the run that starts at r0: the next boundary bit after r0
            int r1 = IG_CH;
#pragma unroll
            for (int g = IG_NSTAGE - 1; g >= 0; --g) {
                uint32_t m = bnd[g];
                const int lo = r0 + 1 - g * 32;        // first bit of this word that lies after r0
                if (lo >= 32) m = 0u;
                else if (lo > 0) m &= 0xffffffffu << lo;
                if (m) r1 = g * 32 + __ffs(m) - 1;     // lower words are visited last: smallest wins
            }
            const char* rp = my_rec + r0 * STRIDE;
            const int S = IG_HDR_S(*reinterpret_cast<const uint32_t*>(rp + 8));
            if (S != 0) {
                const int s2 = S * S;
                const int n_pass = (s2 + 32 * IG_RMAX - 1) / (32 * IG_RMAX);
                const int R = (s2 + 32 * n_pass - 1) / (32 * n_pass);   // points per lane, <= IG_RMAX
                for (int pass = 0; pass < n_pass; ++pass) {
                    const int q0 = pass * 32 * R + lane;
                    switch (R) {
#define IG_CASE(r) case r: n_commit += grid_run<NPOL, r, COUNT>(rp, r1 - r0, S, q0, grid_ch, bank, N); break;
                        IG_CASE(1) IG_CASE(2)
#if IG_RMAX >= 3
                        IG_CASE(3)
#endif
#if IG_RMAX >= 4
                        IG_CASE(4)
#endif
#if IG_RMAX >= 5
                        IG_CASE(5)
#endif
#if IG_RMAX >= 6
                        IG_CASE(6)
#endif
#if IG_RMAX >= 8
                        IG_CASE(7) IG_CASE(8)
#endif
#undef IG_CASE
                        default: break;
                    }
                }
            }
            r0 = r1;
        }
        phase ^= 1u;
    }
    if constexpr (COUNT) {
        n_commit = __reduce_add_sync(0xffffffffu, n_commit);
        if (lane == 0 && n_commit) atomicAdd(commits, (unsigned long long)n_commit);
    }
}

int ig_launch_gridder(ig_ctx* c, const char* records, const uint32_t* chunk_smax, long long nrb, int nchan) {
    const long long n_chunks = nrb * nchan;
    if (n_chunks == 0) return 0;
    if (n_chunks >= (1ll << 32) - 65536) { c->err = "too many work items"; return -1; }
    IG_CUDA_OK(c, cudaMemsetAsync(&c->d_acc->ticket, 0, sizeof(unsigned), c->stream));
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    int per_sm = IG_GRID_CTAS_PER_SM;
    long long want = (n_chunks + IG_GRID_WARPS - 1) / IG_GRID_WARPS;
    unsigned ctas = (unsigned)(want < (long long)sms * per_sm ? want : (long long)sms * per_sm);
    dim3 g(ctas), b(IG_GRID_WARPS * 32);
    const bool two_phase = n_chunks < 200ll * ctas * IG_GRID_WARPS && n_chunks < (1ll << 30);   // fewer than ~200 items per warp
#define IG_LAUNCH(P, C) k_gridder<P, C><<<g, b, 0, c->stream>>>(records, chunk_smax, (unsigned)nrb, (unsigned)nchan, c->grid, c->d_bank, c->prm.N, &c->d_acc->ticket, &c->d_acc->commits, c->per_channel ? (size_t)c->prm.N * c->prm.N * c->prm.npol * 2 : (size_t)0, two_phase)
    if (c->count_commits) {
        switch (c->prm.npol) { case 1: IG_LAUNCH(1, true); break; case 2: IG_LAUNCH(2, true); break; default: IG_LAUNCH(4, true); break; }
    } else {
        switch (c->prm.npol) { case 1: IG_LAUNCH(1, false); break; case 2: IG_LAUNCH(2, false); break; default: IG_LAUNCH(4, false); break; }
    }
#undef IG_LAUNCH
    IG_CUDA_OK(c, cudaGetLastError());
    return 1;
}
