// ig_api.cu - the C ABI of include/ig.h: argument checks, buffer carving, launch order.
#include <math.h>
#include <string.h>
#include "ig_internal.h"

namespace {
ig_status fail(ig_ctx* c, ig_status s, const std::string& m) { if (c) c->err = m; return s; }

// layout of bank_dev: [IgAccum][per-channel normalisers][planes P][zeta P*beta^2][K data]
size_t bank_head_bytes(const ig_ctx* c) {
    size_t b2 = (size_t)c->prm.beta * c->prm.beta;
    return ig_align(sizeof(IgAccum)) + ig_align((size_t)IG_MAX_CHAN_GRIDS * 4 * 8) + ig_align((size_t)c->prm.P * sizeof(IgPlaneEntry)) +
           ig_align((size_t)c->prm.P * b2 * 8);
}
size_t bank_elems_of(const ig_ctx* c, const int* table) {
    size_t b2 = (size_t)c->prm.beta * c->prm.beta, e = 0;
    for (int p = 0; p < c->prm.P; ++p) {
        size_t S = table ? (size_t)table[p] : (size_t)c->max_support;
        e += S * S * b2;
    }
    return e;
}
bool table_ok(const ig_ctx* c, const int* t) {
    for (int p = 0; p < c->prm.P; ++p)
        if (t[p] < 1 || t[p] > c->max_support || (t[p] & 1) == 0) return false;
    return true;
}
struct GridLayout { size_t freqs, perm, sort, smax, gcount, tile_count, tile_off, tile_cur, plan_hdr, plan_scratch, items, records, entries, total; long long nrb, n_chunks; };
GridLayout grid_layout(const ig_ctx* c, long long nrow, int nchan) {
    GridLayout L{};
    L.nrb = (nrow + IG_CH - 1) / IG_CH;
    L.n_chunks = L.nrb * nchan;
    size_t o = 0;
    L.freqs = o; o += ig_align((size_t)nchan * 8);
    L.perm = o; o += ig_align((size_t)nrow * 4);
    L.sort = o; o += ig_align(ig_sort_scratch_bytes(nrow));
    L.smax = o; o += ig_align((size_t)L.n_chunks * 4);
    L.gcount = o; o += ig_align((size_t)L.n_chunks * 4);          // directly after smax (cleared together)
    // the gather gridder's plan arrays and entry area exist only when a record can reach it (ig_gather_possible):
    // support tables below the threshold need none of them
    const bool gather = ig_gather_possible(c);
    const size_t nt = gather ? ig_gather_bins(c, nchan) : 0;
    L.tile_count = o; o += ig_align(nt * 4);
    L.tile_off = o; o += ig_align(nt * 4);
    L.tile_cur = o; o += ig_align(nt * 4);
    L.plan_hdr = o; o += 256;
    L.plan_scratch = o; o += gather ? ig_align(ig_gather_plan_scratch_bytes(c, nchan)) : 0;
    L.items = o; o += gather ? ig_align(ig_gather_max_items(c, L.n_chunks, nchan) * 16) : 0;
    const size_t rec_bytes = ig_align((size_t)L.n_chunks * IG_CH * ig_rec_stride(c->prm.npol));
    L.records = o; o += rec_bytes;
    L.entries = o; o += gather ? ig_align((size_t)L.n_chunks * IG_CH * (16 + 16 * c->prm.npol)) : 0;   // gather entries: at most every record
    L.total = o;
    return L;
}
// installs the support table: host copies, device plane table; device pointers
int install_table(ig_ctx* c, const int* table) {
    const int P = c->prm.P;
    c->support.assign(table, table + P);
    c->koff.resize(P);
    size_t e = 0, b2 = (size_t)c->prm.beta * c->prm.beta;
    for (int p = 0; p < P; ++p) {
        if (e >= (1ull << 32)) { c->err = "bank larger than 2^32 complex elements"; return -1; }
        c->koff[p] = (uint32_t)e;
        e += (size_t)table[p] * table[p] * b2;
    }
    if (e >= (1ull << 32)) { c->err = "bank larger than 2^32 complex elements"; return -1; }
    c->bank_elems = e;
    if (bank_head_bytes(c) + e * 8 > c->bank_bytes) { c->err = "bank buffer too small (see ig_bank_bytes)"; return -2; }
    std::vector<IgPlaneEntry> pe(P);
    for (int p = 0; p < P; ++p) {
        pe[p].support = table[p];
        pe[p].koff = c->koff[p];
        // floor(2^32/S)+1 does not fit 32 bits for S = 1; 2^32-1 there gives x - umulhi(x, magic) = 1 for x > 0 (0 for
        // x = 0), which k_index turns into c = S - 1 = 0: the right answer, since x mod 1 = 0
        pe[p].magic = table[p] == 1 ? 0xffffffffu : (uint32_t)((1ull << 32) / (unsigned)table[p]) + 1u;
        pe[p].pad_ = 0u;
    }
    IG_CUDA_OK(c, cudaMemcpyAsync(c->d_planes, pe.data(), (size_t)P * sizeof(IgPlaneEntry), cudaMemcpyHostToDevice, c->stream));
    IG_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return 0;
}
}  // namespace

extern "C" {

ig_status ig_create(ig_ctx** out, int grid_n, double cell_rad, int n_wplanes, int oversampling, int max_support,
                    int n_pol) {
    if (!out) return IG_EINVAL;
    *out = nullptr;
    if (grid_n < 16 || grid_n > 32768 || (grid_n & 1)) return IG_EINVAL;
    if (!(cell_rad > 0.0) || !isfinite(cell_rad)) return IG_EINVAL;
    if (n_wplanes < 1 || n_wplanes > (1 << 20)) return IG_EINVAL;
    if (oversampling < 1 || oversampling > 16) return IG_EINVAL;
    if (max_support < 3 || (max_support & 1) == 0 || max_support > grid_n) return IG_EINVAL;
    if (max_support > IG_MAX_SUPPORT) return IG_EUNSUPPORTED;   // record headers carry c, d, S in 9 bits each
    if (n_pol != 1 && n_pol != 2 && n_pol != 4) return IG_EINVAL;
    ig_ctx* c = new (std::nothrow) ig_ctx();
    if (!c) return IG_ENOMEM;
    c->prm.N = grid_n; c->prm.beta = oversampling; c->prm.P = n_wplanes; c->prm.npol = n_pol;
    c->prm.shift = (oversampling + 1) / 2 - 1;
    c->prm.bshift = -1;
    for (int b = 0; b < 5; ++b) if (oversampling == (1 << b)) c->prm.bshift = b;
    c->cell_rad = cell_rad;
    c->du = 1.0 / ((double)grid_n * cell_rad);
    c->prm.ku = (double)oversampling / (IG_C_M_S * c->du);
    c->prm.kw = 0.0;
    c->max_support = max_support;
    *out = c;
    return IG_OK;
}

void ig_destroy(ig_ctx* c) {
    if (!c) return;
    for (auto& t : c->ev) for (auto& e : t) if (e) cudaEventDestroy(e);

    for (auto& e : c->ev_copied) if (e) cudaEventDestroy(e);
    for (auto& e : c->ev_free) if (e) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    delete c;
}

const char* ig_last_error(const ig_ctx* c) { return c ? c->err.c_str() : "null context"; }

size_t ig_grid_bytes(const ig_ctx* c) { return c ? (size_t)c->prm.N * c->prm.N * c->prm.npol * 8 : 0; }
size_t ig_workspace_bytes(const ig_ctx* c, long long nrow, int nchan) {
    if (!c || nrow < 0 || nchan < 1) return 0;
    size_t a = grid_layout(c, nrow, nchan).total, b = ig_bank_scratch_bytes(c);
    return a > b ? a : b;
}
size_t ig_bank_bytes(const ig_ctx* c, const int* table) {
    if (!c) return 0;
    return bank_head_bytes(c) + ig_align(bank_elems_of(c, table) * 8);
}
size_t ig_finalize_workspace_bytes(const ig_ctx* c) { return c ? ig_finalize_scratch_bytes(c) : 0; }
static long long host_slice_rows(const ig_ctx* c, long long nrow);
static size_t host_stage_bytes(const ig_ctx* c, long long rows, int nchan);
size_t ig_host_staging_bytes(const ig_ctx* c, long long nrow, int nchan) {
    if (!c || nrow < 0 || nchan < 1) return 0;
    // what ig_grid_host carves after the first ig_workspace_bytes(): one staging area for an unsliced batch, two
    // (double buffering) when the rows are cut into slices; sized for the current ig_set_host_slices() value
    const long long srows = host_slice_rows(c, nrow);
    const size_t pad = ig_align(ig_workspace_bytes(c, srows, nchan)) - ig_workspace_bytes(c, srows, nchan);
    return pad + (srows < nrow ? 2 : 1) * host_stage_bytes(c, srows, nchan);
}

ig_status ig_bind(ig_ctx* c, void* grid_dev, size_t grid_bytes, void* work_dev, size_t work_bytes, void* bank_dev,
                  size_t bank_bytes, void* cuda_stream) {
    if (!c) return IG_EINVAL;
    if (!grid_dev || !work_dev || !bank_dev) return fail(c, IG_EINVAL, "null buffer");
    if (grid_bytes < ig_grid_bytes(c)) return fail(c, IG_ENOMEM, "grid buffer smaller than ig_grid_bytes()");
    if (bank_bytes < bank_head_bytes(c)) return fail(c, IG_ENOMEM, "bank buffer too small");
    if (((uintptr_t)work_dev | (uintptr_t)bank_dev | (uintptr_t)grid_dev) & 255) return fail(c, IG_EINVAL, "buffers must be 256-byte aligned");
    bool moved = (char*)bank_dev != c->bank_buf;
    c->grid = (float*)grid_dev; c->grid_bytes = grid_bytes;
    c->work = (char*)work_dev; c->work_bytes = work_bytes;
    c->bank_buf = (char*)bank_dev; c->bank_bytes = bank_bytes;
    c->stream = (cudaStream_t)cuda_stream;
    char* p = c->bank_buf;
    c->d_acc = (IgAccum*)p; p += ig_align(sizeof(IgAccum));
    c->d_chan_norm = (double*)p; p += ig_align((size_t)IG_MAX_CHAN_GRIDS * 4 * 8);
    c->d_planes = (IgPlaneEntry*)p; p += ig_align((size_t)c->prm.P * sizeof(IgPlaneEntry));
    c->d_zeta = (double*)p; p += ig_align((size_t)c->prm.P * c->prm.beta * c->prm.beta * 8);
    c->d_bank = (float2*)p;
    if (moved) {
        c->have_bank = false;
        cudaError_t e = cudaMemsetAsync(c->d_acc, 0, ig_align(sizeof(IgAccum)) + (size_t)IG_MAX_CHAN_GRIDS * 4 * 8, c->stream);
        if (e != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_bind: ") + cudaGetErrorString(e));
    }
    for (auto& t : c->ev)
        for (auto& ev : t)
            if (!ev && cudaEventCreate(&ev) != cudaSuccess) return fail(c, IG_ECUDA, "cudaEventCreate failed");

    c->bound = true;
    return IG_OK;
}

static ig_status set_wmax(ig_ctx* c, double w_max) {
    if (c->prm.P > 1 && !(w_max > 0.0)) return fail(c, IG_EINVAL, "w_max must be > 0 with more than one w-plane");
    c->w_max = w_max;
    double pm1 = (double)(c->prm.P - 1);
    c->prm.kw = (c->prm.P > 1 && w_max > 0.0) ? (pm1 * pm1) / (IG_C_M_S * w_max) : 0.0;
    return IG_OK;
}

ig_status ig_build_wkernels(ig_ctx* c, double w_max, const int* table) {
    if (!c) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    ig_status s = set_wmax(c, w_max);
    if (s != IG_OK) return s;
    std::vector<int> detected;
    if (!table) {                       // automatic supports: the thesis's 1e-3 rule (:1114), reading 7
        detected.resize(c->prm.P);
        if (ig_detect_supports(c, c->work, c->work_bytes, detected.data()) < 0)
            return c->err.find("too small") != std::string::npos ? IG_ENOMEM : IG_ECUDA;
        table = detected.data();
    }
    if (!table_ok(c, table)) return fail(c, IG_EINVAL, "supports must be odd and within [1, max_support]");
    int r = install_table(c, table);
    if (r < 0) return r == -2 ? IG_ENOMEM : IG_ECUDA;
    if (ig_launch_bank(c, c->work, c->work_bytes) < 0) return c->err.find("too small") != std::string::npos ? IG_ENOMEM : IG_ECUDA;
    c->have_bank = true;
    return IG_OK;
}

ig_status ig_get_supports(ig_ctx* c, int* table) {
    if (!c || !table) return IG_EINVAL;
    if (!c->have_bank) return fail(c, IG_ESTATE, "no bank");
    for (int p = 0; p < c->prm.P; ++p) table[p] = c->support[p];
    return IG_OK;
}

ig_status ig_debug_set_wkernels(ig_ctx* c, double w_max, const int* table, const float* bank_host, size_t bytes) {
    if (!c || !table || !bank_host) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    if (!table_ok(c, table)) return fail(c, IG_EINVAL, "supports must be odd and within [1, max_support]");
    ig_status s = set_wmax(c, w_max);
    if (s != IG_OK) return s;
    int r = install_table(c, table);
    if (r < 0) return r == -2 ? IG_ENOMEM : IG_ECUDA;
    if (bytes != c->bank_elems * 8) return fail(c, IG_EINVAL, "bank size does not match the support table");
    if (cudaMemcpyAsync(c->d_bank, bank_host, bytes, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return fail(c, IG_ECUDA, "copying the bank failed");
    if (ig_launch_zeta(c) < 0) return IG_ECUDA;
    c->have_bank = true;
    return IG_OK;
}

ig_status ig_debug_get_wkernels(ig_ctx* c, float* bank_host, size_t bytes) {
    if (!c || !bank_host) return IG_EINVAL;
    if (!c->have_bank) return fail(c, IG_ESTATE, "no bank");
    if (bytes != c->bank_elems * 8) return fail(c, IG_EINVAL, "bank size mismatch");
    if (cudaMemcpyAsync(bank_host, c->d_bank, bytes, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return fail(c, IG_ECUDA, std::string("reading the bank failed: ") + cudaGetErrorString(cudaGetLastError()));
    return IG_OK;
}

ig_status ig_grid(ig_ctx* c, const double* uvw, const int* baseline_id, long long nrow, const double* freqs,
                  int nchan, const float* vis, const float* wt) {
    if (!c) return IG_EINVAL;
    if (!c->bound || !c->have_bank) return fail(c, IG_ESTATE, "ig_bind and ig_build_wkernels first");
    if (nrow < 0 || nchan < 1 || !freqs) return fail(c, IG_EINVAL, "bad nrow/nchan/freqs");
    if (c->per_channel && (nchan > IG_MAX_CHAN_GRIDS || (size_t)nchan * ig_grid_bytes(c) > c->grid_bytes))
        return fail(c, IG_ENOMEM, "per-channel grids: the bound grid buffer holds fewer than nchan grids");
    c->launches = 0;
    if (nrow == 0) return IG_OK;
    if (!uvw || !baseline_id || !vis || !wt) return fail(c, IG_EINVAL, "null input");
    if (((uintptr_t)uvw & 7) || ((uintptr_t)baseline_id & 3) || (((uintptr_t)vis | (uintptr_t)wt) & (c->prm.npol == 4 ? 15 : 3)))
        return fail(c, IG_EINVAL, "misaligned input (n_pol = 4: vis and weights must be 16-byte aligned)");
    GridLayout L = grid_layout(c, nrow, nchan);
    if (L.total > c->work_bytes) return fail(c, IG_ENOMEM, "work buffer smaller than ig_workspace_bytes()");
    double* d_freqs = (double*)(c->work + L.freqs);
    uint32_t* perm = (uint32_t*)(c->work + L.perm);
    uint32_t* smax = (uint32_t*)(c->work + L.smax);
    char* records = c->work + L.records;
    cudaEvent_t* ev = c->ev[c->n_timed % IG_TIMING_RING];
    cudaError_t e = cudaEventRecord(ev[0], c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_freqs, freqs, (size_t)nchan * 8, cudaMemcpyHostToDevice, c->stream);
    if (e != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_grid: ") + cudaGetErrorString(e));
    double fref = 0;
    for (int k = 0; k < nchan; ++k) fref += freqs[k] / nchan;
    int n = ig_launch_sort_rows(c, uvw, baseline_id, nrow, fref, perm, c->work + L.sort, ig_sort_scratch_bytes(nrow));
    if (n < 0) return IG_ECUDA;
    c->launches += n;
    uint32_t* gcount = (uint32_t*)(c->work + L.gcount);
    uint32_t* tile_count = (uint32_t*)(c->work + L.tile_count);
    const bool any_gather = ig_gather_possible(c);
    const int gather_min = any_gather ? c->gather_min : (IG_MAX_SUPPORT + 1);
    n = ig_launch_index(c, uvw, perm, nrow, d_freqs, nchan, vis, wt, records, smax, gcount, tile_count, gather_min);
    if (n < 0) return IG_ECUDA;
    c->launches += n;
    cudaEventRecord(ev[1], c->stream);
    n = ig_launch_gridder(c, records, smax, L.nrb, nchan);
    if (n < 0) return IG_ECUDA;
    c->launches += n;
    cudaEventRecord(ev[2], c->stream);
    if (any_gather) {
        n = ig_launch_gather(c, records, gcount, L.n_chunks, nchan, tile_count, (uint32_t*)(c->work + L.tile_off),
                             (uint32_t*)(c->work + L.tile_cur), (uint4*)(c->work + L.items), (uint32_t*)(c->work + L.plan_hdr),
                             c->work + L.entries, (unsigned long long*)(c->work + L.plan_scratch));
        if (n < 0) return IG_ECUDA;
        c->launches += n;
    }
    cudaEventRecord(ev[3], c->stream);
    c->n_timed += 1;
    return IG_OK;
}

// Host entry point: the rows are cut into `host_slices` slices; slice k+1 is copied (second stream, double
// buffered staging inside work_dev) while slice k is ordered, indexed and gridded. ig_grid is additive, so the
// slices need no merge step. The copies overlap the kernels only if the caller's buffers are pinned.
static long long host_slice_rows(const ig_ctx* c, long long nrow) {
    int k = c->host_slices;
    if (nrow < (1 << 16)) k = 1;
    if (k == 1) return nrow;                         // unsliced: ig_grid takes a partial last row block
    long long r = (nrow + k - 1) / k;
    r = (r + IG_CH - 1) / IG_CH * IG_CH;             // whole row blocks
    return r < nrow ? r : nrow;
}
static size_t host_stage_bytes(const ig_ctx* c, long long rows, int nchan) {
    size_t rec = (size_t)rows * nchan * c->prm.npol;
    return ig_align((size_t)rows * 24) + ig_align((size_t)rows * 4) + ig_align(rec * 8) + ig_align(rec * 4);
}

ig_status ig_set_host_slices(ig_ctx* c, int n) {
    if (!c || n < 1 || n > 1024) return IG_EINVAL;
    c->host_slices = n;
    return IG_OK;
}

ig_status ig_grid_host(ig_ctx* c, const double* uvw, const int* baseline_id, long long nrow, const double* freqs,
                       int nchan, const float* vis, const float* wt) {
    if (!c) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    if (nrow < 0 || nchan < 1) return fail(c, IG_EINVAL, "bad nrow/nchan");
    if (nrow == 0) return IG_OK;
    if (!uvw || !baseline_id || !vis || !wt) return fail(c, IG_EINVAL, "null input");
    const long long srows = host_slice_rows(c, nrow);
    const size_t base = ig_align(ig_workspace_bytes(c, srows, nchan));
    const size_t stage = host_stage_bytes(c, srows, nchan);
    const int nbuf = srows < nrow ? 2 : 1;
    if (base + nbuf * stage > c->work_bytes) return fail(c, IG_ENOMEM, "work buffer smaller than ig_workspace_bytes(slice rows) + ig_host_staging_bytes()");
    if (!c->copy_stream) {
        if (cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return fail(c, IG_ECUDA, "cannot create the copy stream");
        for (auto& e : c->ev_copied) cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
        for (auto& e : c->ev_free) cudaEventCreateWithFlags(&e, cudaEventDisableTiming);
    }
    // the staging area may still be in use by work queued earlier on the bound stream
    cudaError_t e = cudaEventRecord(c->ev_free[0], c->stream);
    if (e == cudaSuccess) e = cudaEventRecord(c->ev_free[1], c->stream);
    if (e != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_grid_host: ") + cudaGetErrorString(e));
    const size_t vrow = (size_t)nchan * c->prm.npol;     // visibilities per row
    int launches = 0, k = 0;
    for (long long r0 = 0; r0 < nrow; r0 += srows, ++k) {
        const long long rows = (nrow - r0 < srows) ? nrow - r0 : srows;
        const int b = k & 1;
        char* p = c->work + base + (size_t)b * stage;
        double* d_uvw = (double*)p; p += ig_align((size_t)srows * 24);
        int* d_bl = (int*)p; p += ig_align((size_t)srows * 4);
        float* d_vis = (float*)p; p += ig_align((size_t)srows * vrow * 8);
        float* d_wt = (float*)p;
        e = cudaStreamWaitEvent(c->copy_stream, c->ev_free[b], 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_uvw, uvw + 3 * r0, (size_t)rows * 24, cudaMemcpyHostToDevice, c->copy_stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_bl, baseline_id + r0, (size_t)rows * 4, cudaMemcpyHostToDevice, c->copy_stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_vis, vis + (size_t)r0 * vrow * 2, (size_t)rows * vrow * 8, cudaMemcpyHostToDevice, c->copy_stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_wt, wt + (size_t)r0 * vrow, (size_t)rows * vrow * 4, cudaMemcpyHostToDevice, c->copy_stream);
        if (e == cudaSuccess) e = cudaEventRecord(c->ev_copied[b], c->copy_stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(c->stream, c->ev_copied[b], 0);
        if (e != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_grid_host: ") + cudaGetErrorString(e));
        ig_status st = ig_grid(c, d_uvw, d_bl, rows, freqs, nchan, d_vis, d_wt);
        if (st != IG_OK) return st;
        launches += c->launches;
        e = cudaEventRecord(c->ev_free[b], c->stream);
        if (e != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_grid_host: ") + cudaGetErrorString(e));
    }
    c->launches = launches;
    return IG_OK;
}

ig_status ig_set_gather_min_support(ig_ctx* c, int s) {
    if (!c || s < 1) return IG_EINVAL;
    c->gather_min = s;
    return IG_OK;
}

ig_status ig_set_sort_tile_shift(ig_ctx* c, int shift) {
    if (!c || (shift != 0 && (shift < 5 || shift > 15))) return IG_EINVAL;
    c->tile_shift = shift;
    return IG_OK;
}

ig_status ig_set_per_channel_grids(ig_ctx* c, int on) {
    if (!c) return IG_EINVAL;
    c->per_channel = on != 0;
    return IG_OK;
}

ig_status ig_finalize_channel(ig_ctx* c, int channel, float* image_dev, double* norm_host) {
    if (!c || !image_dev || channel < 0 || channel >= IG_MAX_CHAN_GRIDS) return IG_EINVAL;
    if (!c->bound || !c->have_bank || !c->per_channel) return fail(c, IG_ESTATE, "per-channel grids are not in use");
    if ((size_t)(channel + 1) * ig_grid_bytes(c) > c->grid_bytes) return fail(c, IG_EINVAL, "no such channel grid");
    int r = ig_run_finalize(c, channel, image_dev, norm_host, c->stokes);
    if (r == -2) return IG_ENOMEM;
    return r < 0 ? IG_ECUDA : IG_OK;
}

ig_status ig_finalize(ig_ctx* c, float* image_dev, double* norm_host) {
    if (!c || !image_dev) return IG_EINVAL;
    if (!c->bound || !c->have_bank) return fail(c, IG_ESTATE, "nothing to finalise");
    if (c->per_channel) return fail(c, IG_ESTATE, "per-channel grids: use ig_finalize_channel");
    int r = ig_run_finalize(c, -1, image_dev, norm_host, c->stokes);
    if (r == -2) return IG_ENOMEM;
    return r < 0 ? IG_ECUDA : IG_OK;
}

ig_status ig_set_stokes_output(ig_ctx* c, int on) {
    if (!c) return IG_EINVAL;
    c->stokes = on != 0;
    return IG_OK;
}

ig_status ig_get_stats(ig_ctx* c, long long* g, long long* d, long long* u) {
    if (!c) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    IgAccum a;
    if (cudaMemcpyAsync(&a, c->d_acc, sizeof(a), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return fail(c, IG_ECUDA, std::string("ig_get_stats: ") + cudaGetErrorString(cudaGetLastError()));
    if (g) *g = (long long)a.gridded;
    if (d) *d = (long long)a.dropped;
    if (u) *u = (long long)a.updates;
    return IG_OK;
}

ig_status ig_set_commit_counting(ig_ctx* c, int on) {
    if (!c) return IG_EINVAL;
    c->count_commits = on != 0;
    return IG_OK;
}

ig_status ig_set_compression(ig_ctx* c, int on) {
    if (!c) return IG_EINVAL;
    c->compress = on != 0;
    return IG_OK;
}

ig_status ig_get_compressed(ig_ctx* c, long long* n) {
    if (!c || !n) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    IgAccum a;
    if (cudaMemcpyAsync(&a, c->d_acc, sizeof(a), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return fail(c, IG_ECUDA, std::string("ig_get_compressed: ") + cudaGetErrorString(cudaGetLastError()));
    *n = (long long)a.merged;
    return IG_OK;
}

ig_status ig_get_commits(ig_ctx* c, long long* n) {
    if (!c || !n) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    IgAccum a;
    if (cudaMemcpyAsync(&a, c->d_acc, sizeof(a), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
        cudaStreamSynchronize(c->stream) != cudaSuccess)
        return fail(c, IG_ECUDA, std::string("ig_get_commits: ") + cudaGetErrorString(cudaGetLastError()));
    *n = (long long)a.commits;
    return IG_OK;
}

ig_status ig_get_timing(ig_ctx* c, int calls_back, float* ingest_ms, float* gridder_ms) {
    if (!c || calls_back < 0 || calls_back >= IG_TIMING_RING) return IG_EINVAL;
    if (c->n_timed <= calls_back) return fail(c, IG_ESTATE, "no such timed ig_grid call");
    cudaEvent_t* ev = c->ev[(c->n_timed - 1 - calls_back) % IG_TIMING_RING];
    if (cudaEventSynchronize(ev[3]) != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_get_timing: ") + cudaGetErrorString(cudaGetLastError()));
    float a = 0, b = 0;
    cudaEventElapsedTime(&a, ev[0], ev[1]);
    cudaEventElapsedTime(&b, ev[1], ev[3]);
    if (ingest_ms) *ingest_ms = a;
    if (gridder_ms) *gridder_ms = b;
    return IG_OK;
}

ig_status ig_get_gridder_split(ig_ctx* c, int calls_back, float* window_ms, float* gather_ms) {
    if (!c || calls_back < 0 || calls_back >= IG_TIMING_RING) return IG_EINVAL;
    if (c->n_timed <= calls_back) return fail(c, IG_ESTATE, "no such timed ig_grid call");
    cudaEvent_t* ev = c->ev[(c->n_timed - 1 - calls_back) % IG_TIMING_RING];
    if (cudaEventSynchronize(ev[3]) != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_get_gridder_split: ") + cudaGetErrorString(cudaGetLastError()));
    float a = 0, b = 0;
    cudaEventElapsedTime(&a, ev[1], ev[2]);
    cudaEventElapsedTime(&b, ev[2], ev[3]);
    if (window_ms) *window_ms = a;
    if (gather_ms) *gather_ms = b;
    return IG_OK;
}

ig_status ig_reset_accumulators(ig_ctx* c) {
    if (!c) return IG_EINVAL;
    if (!c->bound) return fail(c, IG_ESTATE, "ig_bind first");
    if (cudaMemsetAsync(c->d_acc, 0, ig_align(sizeof(IgAccum)) + (size_t)IG_MAX_CHAN_GRIDS * 4 * 8, c->stream) != cudaSuccess) return fail(c, IG_ECUDA, "memset failed");
    return IG_OK;
}

int ig_last_launches(const ig_ctx* c) { return c ? c->launches : 0; }

ig_status ig_debug_indices(ig_ctx* c, const double* uvw, long long nrow, const double* freqs, int nchan, int* X, int* Y,
                           int* ou, int* ov, int* pl, int* fl) {
    if (!c || !uvw || !freqs || nrow < 0 || nchan < 1) return IG_EINVAL;
    if (!c->bound || !c->have_bank) return fail(c, IG_ESTATE, "ig_bind and a support table first");
    if ((size_t)nchan * 8 > c->work_bytes) return fail(c, IG_ENOMEM, "work buffer too small");
    double* d_freqs = (double*)c->work;
    if (cudaMemcpyAsync(d_freqs, freqs, (size_t)nchan * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        return fail(c, IG_ECUDA, "copying freqs failed");
    if (ig_launch_debug_index(c, uvw, nrow, d_freqs, nchan, X, Y, ou, ov, pl, fl) < 0) return IG_ECUDA;
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return fail(c, IG_ECUDA, std::string("ig_debug_indices: ") + cudaGetErrorString(e));
    return IG_OK;
}

ig_status ig_debug_taper(const double* eta, int n, double* psi) {
    if (!eta || !psi || n < 0) return IG_EINVAL;
    ig_taper_eval(eta, n, psi);
    return IG_OK;
}

}  // extern "C"
