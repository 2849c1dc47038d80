// ig_ingest.cu - steps A1 (index precompute) and A3 (filter + work items).
//
// A1 follows PreProcessUVW (sec 4.4.5): per record the conjugate
// flag (eq 4.10), the cell and sub-cell offset (eq 4.1-4.2 :1076-1091 on the nearest
// oversampled sample, eq 2.11-2.13 :546-564), the w-plane (:633,:1068), the Romein
// position tuple (eq 4.7 :1325-1331: a = X-h, c = -a mod S, d = -(Y-h) mod S) and the
// kernel pointer z_i; plus the weighted, conjugated visibility (eq 4.16 :1544-1548) and
// the normaliser / statistics terms (eq 4.5, eq 4.17). All coordinate arithmetic is
// fp64 with explicitly rounded multiplies (no FMA contraction) so that the integers
// are bit-identical to an IEEE CPU evaluation of the same formulas (DESIGN.md C.1).
//
// A3: the thesis compacts the record stream and builds a plan of equal-support chunks
// (Alg 4.2-4.3, eq 4.8). Here the layout is data-independent instead: records are written
// at (row block, channel, row in block), every IG_CH consecutive records are one work
// item, dropped records stay as 16-byte "skip" headers (S = 0), and the only plan datum
// is the largest support per item. No scan, no host round trip.
#include "ig_internal.h"
#ifndef IG_INDEX_CG
#define IG_INDEX_CG 2        // channels whose visibilities are requested together (two such groups are in flight)
#endif
#ifndef IG_INDEX_CTAS
#define IG_INDEX_CTAS 4      // resident CTAs per SM the register allocation aims at
#endif

struct IgIndex { int X, Y, ou, ov, p, S, on; };

__device__ __forceinline__ long long floordiv_ll(long long a, long long b) {
    long long q = a / b;
    if ((a % b != 0) && ((a < 0) != (b < 0))) q -= 1;
    return q;
}

// um, vm, wm already flipped so that wm >= 0
__device__ __forceinline__ IgIndex ig_index_one(const IgParams& P, const IgPlaneEntry* __restrict__ planes,
                                                double um, double vm, double wm, double nu) {
    IgIndex r;
    double fu = __dmul_rn(__dmul_rn(um, nu), P.ku);
    double fv = __dmul_rn(__dmul_rn(vm, nu), P.ku);
    double wl = __dmul_rn(wm, nu);
    // a non-finite coordinate has no cell: the record is dropped (reading 20). Decided before any integer conversion
    // or table lookup; the tuple of such a record is all zero apart from the conj bit
    const bool finite = isfinite(fu) && isfinite(fv) && isfinite(wl);
    if (!finite) { fu = 0.0; fv = 0.0; wl = 0.0; }
    long long U = (long long)ceil(__dsub_rn(fu, 0.5));   // nearest sample, ties towards -inf
    long long V = (long long)ceil(__dsub_rn(fv, 0.5));
    long long x, y;                                      // -du/2 < delta <= du/2 (eq 4.2)
    const long long lim32 = 1ll << 30;
    if (U > -lim32 && U < lim32 && V > -lim32 && V < lim32) {
        // every record near the grid: the same floor division in 32 bits (a 64-bit divide is ~80 instructions)
        const int nu_ = (int)U + P.shift, nv_ = (int)V + P.shift;
        int qx, qy;
        if (P.bshift >= 0) {              // beta a power of two: the arithmetic shift is the floor division
            qx = nu_ >> P.bshift; qy = nv_ >> P.bshift;
        } else {
            qx = nu_ / P.beta; qy = nv_ / P.beta;
            if (nu_ - qx * P.beta < 0) qx -= 1;
            if (nv_ - qy * P.beta < 0) qy -= 1;
        }
        x = qx; y = qy;
    } else {
        x = floordiv_ll(U + P.shift, P.beta);
        y = floordiv_ll(V + P.shift, P.beta);
    }
    r.ou = (int)(U - x * P.beta);
    r.ov = (int)(V - y * P.beta);
    int p = 0;
    if (P.P > 1) {
        double sp = floor(__dadd_rn(__dsqrt_rn(__dmul_rn(wl, P.kw)), 0.5));
        p = sp >= (double)(P.P - 1) ? P.P - 1 : (int)sp;
    }
    r.p = p;
    r.S = planes[p].support;
    long long h = (r.S - 1) / 2;
    long long Xc = x + P.N / 2, Yc = y + P.N / 2;
    r.on = (Xc - h >= 0) && (Xc + h <= P.N - 1) && (Yc - h >= 0) && (Yc + h <= P.N - 1);
    if (!finite) { r.on = 0; r.ou = r.ov = 0; Xc = Yc = 0; r.p = 0; r.S = planes[0].support; }
    const long long lim = 1ll << 30;
    Xc = Xc < -lim ? -lim : (Xc > lim ? lim : Xc);
    Yc = Yc < -lim ? -lim : (Yc > lim ? lim : Yc);
    r.X = (int)Xc; r.Y = (int)Yc;
    return r;
}

// One CTA = one row block of IG_CH sorted rows; thread t = row rb*IG_CH + t; loop over channels.
// Record at place ((rb*nchan + c)*IG_CH + t): 16-byte header {pix_base, kbase, z = c | d<<9 | S<<18 | flags (ig_internal.h), plane}
// followed by npol complex32 pairs (stride 48 B for 4 pol, else 32 B).
template <int NPOL>
__global__ void __launch_bounds__(IG_CH, IG_INDEX_CTAS)
k_index(IgParams P, const IgPlaneEntry* __restrict__ planes, const double* __restrict__ zeta,
        const double* __restrict__ uvw, const uint32_t* __restrict__ perm, long long nrow,
        const double* __restrict__ freqs, int nchan, const float* __restrict__ vis,
        const float* __restrict__ wt, char* __restrict__ records, uint32_t* __restrict__ chunk_smax,
        IgAccum* __restrict__ acc, bool compress, double* __restrict__ chan_norm,
        uint32_t* __restrict__ gcount, uint32_t* __restrict__ tile_count, int gather_min, int tiles_x) {
    constexpr int STRIDE = NPOL == 4 ? 48 : 32;
    const long long rb = blockIdx.x;
    const int t = threadIdx.x, lane = t & 31;
    const long long j = rb * IG_CH + t;
    const bool live = j < nrow;
    long long row = 0;
    double um = 0, vm = 0, wm = 0;
    int conj = 0;
    if (live) {
        row = perm[j];
        um = uvw[3 * row]; vm = uvw[3 * row + 1]; wm = uvw[3 * row + 2];
        conj = wm < 0.0;
        if (conj) { um = -um; vm = -vm; wm = -wm; }
    }
    double nsum[NPOL];
#pragma unroll
    for (int q = 0; q < NPOL; ++q) nsum[q] = 0.0;
    unsigned long long n_grid = 0, n_drop = 0, n_upd = 0, n_merged = 0;

    // Channels are taken two at a time, and the visibilities and weights of the NEXT pair are requested before the
    // current pair is worked on (two register buffers, loop unrolled by two pairs): a thread's loads are then in
    // flight all the time instead of only between two ~350-instruction record bodies (ncu: 45 % of the warp time
    // was spent waiting for them).
    constexpr int CG = IG_INDEX_CG;
    float4 pre_a[2][CG], pre_b[2][CG], pre_w[2][CG];
    auto prefetch = [&](int buf, int c0) {
        if constexpr (NPOL == 4) {
#pragma unroll
            for (int k = 0; k < CG; ++k) {
                if (live && c0 + k < nchan) {
                    const float* vp = vis + ((size_t)row * nchan + c0 + k) * 8;
                    pre_a[buf][k] = __ldg(reinterpret_cast<const float4*>(vp));
                    pre_b[buf][k] = __ldg(reinterpret_cast<const float4*>(vp + 4));
                    pre_w[buf][k] = __ldg(reinterpret_cast<const float4*>(wt + ((size_t)row * nchan + c0 + k) * 4));
                }
            }
        }
    };
    prefetch(0, 0);
    for (int c00 = 0; c00 < nchan; c00 += 2 * CG) {
#pragma unroll
     for (int half = 0; half < 2; ++half) {
      const int c0 = c00 + half * CG;
      if (c0 >= nchan) break;
      prefetch(half ^ 1, c0 + CG);
#pragma unroll
      for (int k = 0; k < CG; ++k) {
        const int c = c0 + k;
        if (c >= nchan) break;
        const long long chunk = rb * nchan + c;
        char* rec = records + ((size_t)chunk * IG_CH + t) * STRIDE;
        uint4 hdr = make_uint4(0u, 0u, 0u, 0u);
        float v[2 * NPOL];
#pragma unroll
        for (int q = 0; q < 2 * NPOL; ++q) v[q] = 0.f;
        int S = 0;
        bool is_g = false;                // large support: goes to the gather gridder (ig_gather.cu)
        uint32_t g_tile = 0;
        double cn[NPOL];                  // this record's normaliser terms (per-channel grid mode)
#pragma unroll
        for (int q = 0; q < NPOL; ++q) cn[q] = 0.0;
        if (live) {
            IgIndex ix = ig_index_one(P, planes, um, vm, wm, freqs[c]);
            const float* vp = vis + ((size_t)row * nchan + c) * (2 * NPOL);
            const float* wp = wt + ((size_t)row * nchan + c) * NPOL;
            float w[NPOL];
            bool any = false;
            if constexpr (NPOL == 4) {
                const float4 w4 = pre_w[half][k];
                w[0] = w4.x; w[1] = w4.y; w[2] = w4.z; w[3] = w4.w;
                const float4 a = pre_a[half][k], b = pre_b[half][k];
                (void)vp; (void)wp;
                v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
            } else {
#pragma unroll
                for (int q = 0; q < NPOL; ++q) { w[q] = wp[q]; v[2 * q] = vp[2 * q]; v[2 * q + 1] = vp[2 * q + 1]; }
            }
#pragma unroll
            for (int q = 0; q < NPOL; ++q) any |= (w[q] != 0.f);
            if (ix.on && any) {
                S = ix.S;
                const int h = (S - 1) / 2;
                const int a0 = ix.X - h, b0 = ix.Y - h;
                // (-a0) mod S and (-b0) mod S without integer division: a0, b0 in [0, N), N <= 32768
                const uint32_t magic = planes[ix.p].magic;
                const int ra = a0 - (int)__umulhi((uint32_t)a0, magic) * S, rb2 = b0 - (int)__umulhi((uint32_t)b0, magic) * S;
                const int cm = ra ? S - ra : 0, dm = rb2 ? S - rb2 : 0;
                const uint32_t tab = (uint32_t)((ix.ov + P.shift) * P.beta + (ix.ou + P.shift));
                hdr.y = planes[ix.p].koff + tab * (uint32_t)(S * S);
                is_g = S >= gather_min;
                if (is_g) {
                    hdr.x = (uint32_t)a0 | ((uint32_t)b0 << 16);
                    const uint32_t pstore = min((uint32_t)ix.p, IG_HDR_GPLANE);
                    hdr.z = IG_HDR_GATHER | (conj ? IG_HDR_CONJ : 0u) | pstore;
                    hdr.w = (uint32_t)S;
                    // plan bin: (w-plane bucket, origin tile of 32 x 32 pixels)
                    // per-channel grids: the channel selects the grid, tile = channel * tiles + tile (as k_gather_scatter)
                    const uint32_t nt = (uint32_t)(tiles_x * tiles_x), tl = (uint32_t)((b0 >> 5) * tiles_x + (a0 >> 5));
                    g_tile = chan_norm ? ig_gather_bin((int)pstore, P.P, nt * (uint32_t)nchan, (uint32_t)c * nt + tl)
                                       : ig_gather_bin((int)pstore, P.P, nt, tl);
                } else {
                    hdr.x = (uint32_t)(b0 * P.N + a0);
                    hdr.z = IG_HDR_PACK(cm, dm, S) | (conj ? IG_HDR_CONJ : 0u);
                    hdr.w = (uint32_t)ix.p;
                }
                const double z = zeta[(size_t)ix.p * P.beta * P.beta + tab];
#pragma unroll
                for (int q = 0; q < NPOL; ++q) {
                    cn[q] = (double)w[q] * z;
                    nsum[q] += cn[q];                         // eq 4.5
                    v[2 * q] = w[q] * v[2 * q];               // eq 4.16
                    v[2 * q + 1] = conj ? -(w[q] * v[2 * q + 1]) : w[q] * v[2 * q + 1];
                }
                n_grid += 1;
                n_upd += (unsigned long long)(S * S * NPOL);
            } else {
                n_drop += 1;
            }
        }
        // Compression (eq 4.9 :1407-1414, eq 4.16): records that follow one another with
        // the same cell and the same kernel matrix (plane, sub-cell offsets) are summed into the first of the
        // group; the others stay in place, flagged, and the gridder skips them. Groups are found among the 32
        // consecutive rows of a warp (segmented suffix sum by shuffles; warps without a pair skip it).
        if (compress) {
            const uint32_t px = __shfl_up_sync(0xffffffffu, hdr.x, 1), py = __shfl_up_sync(0xffffffffu, hdr.y, 1);
            const uint32_t pz = __shfl_up_sync(0xffffffffu, hdr.z, 1);
            const bool follows = lane > 0 && S > 0 && px == hdr.x && py == hdr.y && pz == hdr.z;
            const uint32_t heads = __ballot_sync(0xffffffffu, !follows);
            if (heads != 0xffffffffu) {
                const uint32_t after = lane == 31 ? 0u : (heads & (0xffffffffu << (lane + 1)));
                const int end = after ? __ffs(after) - 2 : 31;     // last lane of this lane's group
                // segmented suffix sum; groups are mostly pairs, so stop as soon as no group is longer than o
#pragma unroll 1
                for (int o = 1; o < 32; o <<= 1) {
#pragma unroll
                    for (int q = 0; q < 2 * NPOL; ++q) {
                        const float t = __shfl_down_sync(0xffffffffu, v[q], o);
                        if (lane + o <= end) v[q] += t;
                    }
                    if (!__any_sync(0xffffffffu, lane + 2 * o <= end)) break;
                }
                if (follows) {
                    hdr.z |= IG_HDR_MERGED;
                    n_merged += 1;
#pragma unroll
                    for (int q = 0; q < 2 * NPOL; ++q) v[q] = 0.f;
                }
            }
        }
        *reinterpret_cast<uint4*>(rec) = hdr;
        if constexpr (NPOL == 4) {
            *reinterpret_cast<float4*>(rec + 16) = make_float4(v[0], v[1], v[2], v[3]);
            *reinterpret_cast<float4*>(rec + 32) = make_float4(v[4], v[5], v[6], v[7]);
        } else if constexpr (NPOL == 2) {
            *reinterpret_cast<float4*>(rec + 16) = make_float4(v[0], v[1], v[2], v[3]);
        } else {
            *reinterpret_cast<float4*>(rec + 16) = make_float4(v[0], v[1], 0.f, 0.f);
        }
        if (chan_norm) {                  // one grid per channel: eq 4.5 per channel
#pragma unroll
            for (int q = 0; q < NPOL; ++q) {
                double x = cn[q];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
                if (lane == 0 && x != 0.0) atomicAdd(&chan_norm[(size_t)c * 4 + q], x);
            }
        }
        // plan of the gather gridder: marked records per origin tile (warp-aggregated) and per work item
        const bool count_me = is_g && !(hdr.z & IG_HDR_MERGED);
        const uint32_t gm = __ballot_sync(0xffffffffu, count_me);
        if (gm) {
            if (count_me) {
                const uint32_t peers = __match_any_sync(gm, g_tile);
                if (lane == __ffs(peers) - 1) atomicAdd(&tile_count[g_tile], (uint32_t)__popc(peers));
            }
            if (lane == 0) atomicAdd(&gcount[chunk], (uint32_t)__popc(gm));
        }
        unsigned smax = __reduce_max_sync(0xffffffffu, is_g ? 0u : (unsigned)S);
        if (lane == 0 && smax) atomicMax(&chunk_smax[chunk], smax);
      }
     }
    }

    // block reduction of the normaliser and the counters
    __shared__ double sh[IG_CH / 32][NPOL + 4];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int q = 0; q < NPOL; ++q) nsum[q] += __shfl_xor_sync(0xffffffffu, nsum[q], o);
        n_grid += __shfl_xor_sync(0xffffffffu, n_grid, o);
        n_drop += __shfl_xor_sync(0xffffffffu, n_drop, o);
        n_upd += __shfl_xor_sync(0xffffffffu, n_upd, o);
        n_merged += __shfl_xor_sync(0xffffffffu, n_merged, o);
    }
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NPOL; ++q) sh[t >> 5][q] = nsum[q];
        sh[t >> 5][NPOL] = (double)n_grid; sh[t >> 5][NPOL + 1] = (double)n_drop; sh[t >> 5][NPOL + 2] = (double)n_upd;
        sh[t >> 5][NPOL + 3] = (double)n_merged;
    }
    __syncthreads();
    if (t < NPOL + 4) {
        double s = 0;
        for (int w = 0; w < IG_CH / 32; ++w) s += sh[w][t];   // counts < 2^53: exact in fp64
        if (t < NPOL) atomicAdd(&acc->norm[t], s);
        else if (t == NPOL) atomicAdd(&acc->gridded, (unsigned long long)s);
        else if (t == NPOL + 1) atomicAdd(&acc->dropped, (unsigned long long)s);
        else if (t == NPOL + 2) atomicAdd(&acc->updates, (unsigned long long)s);
        else if (s > 0) atomicAdd(&acc->merged, (unsigned long long)s);
    }
}

__global__ void k_debug_index(IgParams P, const IgPlaneEntry* __restrict__ planes, const double* __restrict__ uvw,
                              long long nrow, const double* __restrict__ freqs, int nchan, int* X, int* Y, int* ou,
                              int* ov, int* pl, int* fl) {
    long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nrow * nchan) return;
    long long r = k / nchan;
    int c = (int)(k - r * nchan);
    double um = uvw[3 * r], vm = uvw[3 * r + 1], wm = uvw[3 * r + 2];
    int conj = wm < 0.0;
    if (conj) { um = -um; vm = -vm; wm = -wm; }
    IgIndex ix = ig_index_one(P, planes, um, vm, wm, freqs[c]);
    X[k] = ix.X; Y[k] = ix.Y; ou[k] = ix.ou; ov[k] = ix.ov; pl[k] = ix.p; fl[k] = conj | (ix.on << 1);
}

int ig_launch_index(ig_ctx* c, const double* uvw, const uint32_t* perm, long long nrow, const double* d_freqs,
                    int nchan, const float* vis, const float* wt, char* records, uint32_t* chunk_smax, uint32_t* gcount,
                    uint32_t* tile_count, int gather_min) {
    long long nrb = (nrow + IG_CH - 1) / IG_CH;
    if (nrb == 0) return 0;
    if (nrb > 0x7fffffffll) { c->err = "too many rows"; return -1; }
    // chunk_smax and gcount are neighbours in the work buffer: one memset clears both
    IG_CUDA_OK(c, cudaMemsetAsync(chunk_smax, 0, (size_t)((char*)(gcount + nrb * nchan) - (char*)chunk_smax), c->stream));
    if (gather_min <= IG_MAX_SUPPORT)   // the plan's bin counts exist only when a record can reach the gather gridder (grid_layout)
        IG_CUDA_OK(c, cudaMemsetAsync(tile_count, 0, ig_gather_bins(c, nchan) * 4, c->stream));
    dim3 g((unsigned)nrb), b(IG_CH);
    const int tiles_x = (c->prm.N + 31) / 32;
#define IG_INDEX(P_) k_index<P_><<<g, b, 0, c->stream>>>(c->prm, c->d_planes, c->d_zeta, uvw, perm, nrow, d_freqs, nchan, vis, wt, records, chunk_smax, c->d_acc, c->compress, c->per_channel ? c->d_chan_norm : nullptr, gcount, tile_count, gather_min, tiles_x)
    switch (c->prm.npol) {
        case 1: IG_INDEX(1); break;
        case 2: IG_INDEX(2); break;
        default: IG_INDEX(4); break;
    }
#undef IG_INDEX
    IG_CUDA_OK(c, cudaGetLastError());
    return 1;
}

int ig_launch_debug_index(ig_ctx* c, const double* uvw, long long nrow, const double* d_freqs, int nchan, int* X,
                          int* Y, int* ou, int* ov, int* pl, int* fl) {
    long long n = nrow * nchan;
    if (n == 0) return 0;
    k_debug_index<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->prm, c->d_planes, uvw, nrow, d_freqs, nchan,
                                                                      X, Y, ou, ov, pl, fl);
    IG_CUDA_OK(c, cudaGetLastError());
    return 1;
}
