// ig_finalize.cu - step E (boundary call ig_finalize), Image Finaliser, Algorithm 4.6
// (PAPER.md:1664-1676): inverse FFT per polarisation (the thesis uses cuFFT too, :952),
// then, per pixel, real part / ( N_p * psi(l)psi(m) * sinc(l)sinc(m) ): normaliser eq 4.5,
// taper correction eq 2.9 (:523), sinc of the nearest-sample lookup eq 2.13 (:561-564).
// Transform convention eq 2.8 (:516): img[b][a] = sum grid[Y][X] e^{+j 2 pi ((X-N/2)a + (Y-N/2)b)/N},
// a,b in [-N/2, N/2), i.e. an unnormalised inverse DFT with both origins at index N/2.
// Stokes conversion is not done (formulas absent from the paper).
#include <cufft.h>
#include <math.h>
#include "ig_internal.h"

template <int NPOL>
__global__ void k_fin_extract(const float2* __restrict__ grid, float2* __restrict__ plane, int N, int pol) {
    int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= N) return;
    int sx = (x + N / 2) % N, sy = (y + N / 2) % N;      // ifftshift: origin N/2 -> 0
    // 4 pol: two planes of polarisation pairs [pair][y][x][2]; 1 or 2 pol: [y][x][pol]
    constexpr int PP = NPOL == 4 ? 2 : NPOL;
    const size_t base = NPOL == 4 ? (size_t)(pol >> 1) * N * N * 2 : 0;
    plane[(size_t)y * N + x] = grid[base + ((size_t)sy * N + sx) * PP + (NPOL == 4 ? (pol & 1) : pol)];
}

__global__ void k_fin_write(const float2* __restrict__ plane, float* __restrict__ image, const double* __restrict__ corr,
                            int N, double norm) {
    int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= N) return;
    int sx = (x + N / 2) % N, sy = (y + N / 2) % N;      // fftshift: origin 0 -> N/2
    double d = norm * corr[x] * corr[y];
    float v = plane[(size_t)sy * N + sx].x;
    image[(size_t)y * N + x] = d != 0.0 ? (float)((double)v / d) : 0.f;
}

static size_t fft_work_bytes(int N) {
    size_t ws = 0;
    if (cufftEstimate2d(N, N, CUFFT_C2C, &ws) != CUFFT_SUCCESS) ws = (size_t)N * N * 8;
    return ws + ws / 8 + (1 << 20);     // the estimate may be below what the made plan asks for
}

size_t ig_finalize_scratch_bytes(const ig_ctx* c) {
    size_t N = c->prm.N;
    return ig_align(N * N * 8) + ig_align(N * 8) + ig_align(fft_work_bytes((int)N));
}

int ig_run_finalize(ig_ctx* c, int channel, float* image, double* norm_host) {
    const int N = c->prm.N, npol = c->prm.npol;
    if (c->work_bytes < ig_finalize_scratch_bytes(c)) { c->err = "work buffer too small for ig_finalize"; return -2; }
    IgAccum acc;
    IG_CUDA_OK(c, cudaMemcpyAsync(&acc, c->d_acc, sizeof(acc), cudaMemcpyDeviceToHost, c->stream));
    IG_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    const float2* grid = (const float2*)c->grid;
    if (channel >= 0) {                 // one grid per channel: its own grid and normaliser
        grid += (size_t)channel * N * N * npol;
        IG_CUDA_OK(c, cudaMemcpyAsync(acc.norm, c->d_chan_norm + (size_t)channel * 4, 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        IG_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    }
    if (norm_host) for (int q = 0; q < npol; ++q) norm_host[q] = acc.norm[q];

    float2* plane = (float2*)c->work;
    double* d_corr = (double*)(c->work + ig_align((size_t)N * N * 8));
    char* fft_ws = (char*)d_corr + ig_align((size_t)N * 8);
    size_t fft_ws_bytes = c->work_bytes - (size_t)(fft_ws - c->work);

    std::vector<double> eta(N), corr(N);
    for (int i = 0; i < N; ++i) eta[i] = 2.0 * (double)(i - N / 2) / (double)N;
    ig_taper_eval(eta.data(), N, corr.data());
    for (int i = 0; i < N; ++i) {
        double x = M_PI * (double)(i - N / 2) / ((double)N * c->prm.beta);
        corr[i] *= (x == 0.0) ? 1.0 : sin(x) / x;
    }
    IG_CUDA_OK(c, cudaMemcpyAsync(d_corr, corr.data(), (size_t)N * 8, cudaMemcpyHostToDevice, c->stream));

    cufftHandle plan;
    size_t need = 0;
    if (cufftCreate(&plan) != CUFFT_SUCCESS) { c->err = "cufftCreate failed"; return -1; }
    cufftSetAutoAllocation(plan, 0);
    if (cufftMakePlan2d(plan, N, N, CUFFT_C2C, &need) != CUFFT_SUCCESS) { cufftDestroy(plan); c->err = "cufftMakePlan2d failed"; return -1; }
    if (need > fft_ws_bytes) { cufftDestroy(plan); c->err = "work buffer too small for the FFT plan"; return -2; }
    cufftSetWorkArea(plan, fft_ws);
    cufftSetStream(plan, c->stream);
    int launches = 0;
    dim3 g((N + 255) / 256, N), b(256);
    for (int q = 0; q < npol; ++q) {
        switch (npol) {
            case 1: k_fin_extract<1><<<g, b, 0, c->stream>>>(grid, plane, N, q); break;
            case 2: k_fin_extract<2><<<g, b, 0, c->stream>>>(grid, plane, N, q); break;
            default: k_fin_extract<4><<<g, b, 0, c->stream>>>(grid, plane, N, q); break;
        }
        if (cufftExecC2C(plan, (cufftComplex*)plane, (cufftComplex*)plane, CUFFT_INVERSE) != CUFFT_SUCCESS) {
            cufftDestroy(plan); c->err = "cufftExecC2C failed"; return -1;
        }
        k_fin_write<<<g, b, 0, c->stream>>>(plane, image + (size_t)q * N * N, d_corr, N, acc.norm[q]);
        launches += 3;
    }
    cudaError_t e = cudaStreamSynchronize(c->stream);
    cufftDestroy(plan);
    if (e != cudaSuccess) { c->err = std::string("ig_finalize: ") + cudaGetErrorString(e); return -1; }
    return launches;
}
