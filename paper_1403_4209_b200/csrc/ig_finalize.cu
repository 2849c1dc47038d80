// ig_finalize.cu - step E (boundary call ig_finalize), Image Finaliser, Algorithm 4.6
// (PAPER.md:1664-1676): inverse FFT per polarisation (the thesis uses cuFFT too, :952),
// then, per pixel, real part / ( N_p * psi(l)psi(m) * sinc(l)sinc(m) ): normaliser eq 4.5,
// taper correction eq 2.9 (:523), sinc of the nearest-sample lookup eq 2.13 (:561-564).
// Transform convention eq 2.8 (:516): img[b][a] = sum grid[Y][X] e^{+j 2 pi ((X-N/2)a + (Y-N/2)b)/N},
// a,b in [-N/2, N/2), i.e. an unnormalised inverse DFT with both origins at index N/2.
// Step 2's Stokes conversion (:1660, :1668; reading 21: linear feeds XX, XY, YX, YY) is ig_finalize_stokes:
// the transform is linear, so the combination of the normalised polarisations is formed on the uv-grid
// (k_fin_combine) and one inverse FFT per Stokes parameter follows.
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

// plane = sum_p coef[p] * grid_p (complex coefficients): one Stokes parameter's uv-grid, normalisers folded into coef
template <int NPOL>
__global__ void k_fin_combine(const float2* __restrict__ grid, float2* __restrict__ plane, int N, float2 c0, float2 c1,
                              float2 c2, float2 c3) {
    int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    if (x >= N) return;
    int sx = (x + N / 2) % N, sy = (y + N / 2) % N;
    const float2 cf[4] = {c0, c1, c2, c3};
    constexpr int PP = NPOL == 4 ? 2 : NPOL;
    float re = 0.f, im = 0.f;
#pragma unroll
    for (int pol = 0; pol < NPOL; ++pol) {
        const size_t base = NPOL == 4 ? (size_t)(pol >> 1) * N * N * 2 : 0;
        const float2 g = grid[base + ((size_t)sy * N + sx) * PP + (NPOL == 4 ? (pol & 1) : pol)];
        re += cf[pol].x * g.x - cf[pol].y * g.y;
        im += cf[pol].x * g.y + cf[pol].y * g.x;
    }
    plane[(size_t)y * N + x] = make_float2(re, im);
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

int ig_run_finalize(ig_ctx* c, int channel, float* image, double* norm_host, bool stokes) {
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
    // Stokes parameter s = sum_p M[s][p] D_p with D_p = img_p / N_p (reading 21); the coefficients carry N_ref / N_p so that
    // the grids keep their scale through the fp32 FFT and k_fin_write divides by N_ref in fp64. N_ref is the largest
    // normaliser in magnitude, so a fully flagged polarisation (N_p = 0, and then an all-zero grid) cannot zero the
    // scale of the others; such a polarisation enters the combinations as D_p = 0 (reading 21)
    double nref = 0.0;
    for (int p = 0; p < npol; ++p) if (fabs(acc.norm[p]) > fabs(nref)) nref = acc.norm[p];
    for (int q = 0; q < npol; ++q) {
        if (stokes && npol > 1) {
            double m[4][2] = {{0, 0}, {0, 0}, {0, 0}, {0, 0}};          // complex coefficient per polarisation
            if (npol == 4) {
                if (q == 0) { m[0][0] = 0.5; m[3][0] = 0.5; }            // I = (XX + YY)/2
                if (q == 1) { m[0][0] = 0.5; m[3][0] = -0.5; }           // Q = (XX - YY)/2
                if (q == 2) { m[1][0] = 0.5; m[2][0] = 0.5; }            // U = (XY + YX)/2
                if (q == 3) { m[1][1] = -0.5; m[2][1] = 0.5; }           // V = (XY - YX)/(2j)
            } else {
                m[0][0] = 0.5; m[1][0] = q == 0 ? 0.5 : -0.5;            // (XX, YY): I, Q
            }
            float2 cf[4];
            for (int p = 0; p < 4; ++p) {
                const double sc = (p < npol && acc.norm[p] != 0.0) ? nref / acc.norm[p] : 0.0;
                cf[p] = make_float2((float)(m[p][0] * sc), (float)(m[p][1] * sc));
            }
            if (npol == 4) k_fin_combine<4><<<g, b, 0, c->stream>>>(grid, plane, N, cf[0], cf[1], cf[2], cf[3]);
            else k_fin_combine<2><<<g, b, 0, c->stream>>>(grid, plane, N, cf[0], cf[1], cf[2], cf[3]);
        } else switch (npol) {
            case 1: k_fin_extract<1><<<g, b, 0, c->stream>>>(grid, plane, N, q); break;
            case 2: k_fin_extract<2><<<g, b, 0, c->stream>>>(grid, plane, N, q); break;
            default: k_fin_extract<4><<<g, b, 0, c->stream>>>(grid, plane, N, q); break;
        }
        if (cufftExecC2C(plan, (cufftComplex*)plane, (cufftComplex*)plane, CUFFT_INVERSE) != CUFFT_SUCCESS) {
            cufftDestroy(plan); c->err = "cufftExecC2C failed"; return -1;
        }
        k_fin_write<<<g, b, 0, c->stream>>>(plane, image + (size_t)q * N * N, d_corr, N, (stokes && npol > 1) ? nref : acc.norm[q]);
        launches += 3;
    }
    cudaError_t e = cudaStreamSynchronize(c->stream);
    cufftDestroy(plan);
    if (e != cudaSuccess) { c->err = std::string("ig_finalize: ") + cudaGetErrorString(e); return -1; }
    return launches;
}
