// ig_bank.cu - step D (boundary call ig_build_wkernels) and the taper.
//
// Convolution Function Generator, Algorithm 4.1: per w-plane the
// image-plane function  f_p(l,m) = psi(l) psi(m) exp(+j 2 pi w_p (sqrt(1-l^2-m^2) - 1))
// (taper x conjugate w-screen, eq 2.14 :580, eq 2.21 :606-615) is sampled on n x n points
// across the field of view, zero padded by the oversampling factor beta and Fourier
// transformed; normalised so that C_0(0,0) = 1 (:1114); then trimmed to the support and
// re-ordered so that every (off_v, off_u) S x S matrix is contiguous (:1100-1108).
// The zero-padded FFT is evaluated here as a partial DFT (only the samples the bank keeps),
// in fp64, as two passes: Gt[b][qu] = sum_a f[b][a] W^(qu a), K = sum_b Gt[b][qu] W^(qv b) / A.
// w_p = w_max (p/(P-1))^2 (:633,:1068). Output complex64.
//
// Taper psi: the prolate-spheroidal gridding function of Schwab that the thesis takes from
// casacore (:1064). The paper prints no coefficients (reading 6), so psi is obtained from its
// defining property: the even eigenfunction with the largest eigenvalue of
//   mu psi(eta) = int_{-1}^{1} (1-t^2)^alpha cos(c eta t) psi(t) dt,  alpha = 1, c = 3 pi.
// Here: Gauss-Legendre nodes by Newton iteration, symmetrised Nystrom matrix, cyclic Jacobi
// eigen-solver, Nystrom extension; psi(0) = 1, psi = 0 for |eta| >= 1.
#include <math.h>
#include <mutex>
#include "ig_internal.h"

namespace {
constexpr int TQ = 80;            // quadrature nodes
constexpr double TC = 9.42477796076937971538793014983850865259;   // 3 pi
struct Taper { double t[TQ], d[TQ], vec[TQ], mu, at0; };
Taper g_taper;
std::once_flag g_taper_once;

void gauss_legendre(int n, double* x, double* w) {
    for (int i = 0; i < n; ++i) {
        double z = cos(M_PI * (i + 0.75) / (n + 0.5)), pp = 1;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1, p2 = 0;
            for (int k = 1; k <= n; ++k) { double p3 = p2; p2 = p1; p1 = ((2.0 * k - 1) * z * p2 - (k - 1.0) * p3) / k; }
            pp = n * (z * p1 - p2) / (z * z - 1);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        x[i] = z; w[i] = 2.0 / ((1 - z * z) * pp * pp);
    }
}

void build_taper() {
    static double A[TQ][TQ], V[TQ][TQ];
    double wq[TQ];
    Taper& T = g_taper;
    gauss_legendre(TQ, T.t, wq);
    for (int i = 0; i < TQ; ++i) T.d[i] = wq[i] * (1.0 - T.t[i] * T.t[i]);
    for (int i = 0; i < TQ; ++i)
        for (int k = 0; k < TQ; ++k) {
            A[i][k] = sqrt(T.d[i]) * cos(TC * T.t[i] * T.t[k]) * sqrt(T.d[k]);
            V[i][k] = i == k;
        }
    for (int sweep = 0; sweep < 60; ++sweep) {       // cyclic Jacobi
        double off = 0;
        for (int i = 0; i < TQ; ++i) for (int k = i + 1; k < TQ; ++k) off += A[i][k] * A[i][k];
        if (off < 1e-30) break;
        for (int p = 0; p < TQ; ++p)
            for (int q = p + 1; q < TQ; ++q) {
                if (fabs(A[p][q]) < 1e-300) continue;
                double th = (A[q][q] - A[p][p]) / (2 * A[p][q]);
                double tt = (th >= 0 ? 1.0 : -1.0) / (fabs(th) + sqrt(th * th + 1));
                double cs = 1 / sqrt(tt * tt + 1), sn = tt * cs;
                for (int k = 0; k < TQ; ++k) {
                    double akp = A[k][p], akq = A[k][q];
                    A[k][p] = cs * akp - sn * akq; A[k][q] = sn * akp + cs * akq;
                }
                for (int k = 0; k < TQ; ++k) {
                    double apk = A[p][k], aqk = A[q][k];
                    A[p][k] = cs * apk - sn * aqk; A[q][k] = sn * apk + cs * aqk;
                }
                for (int k = 0; k < TQ; ++k) {
                    double vkp = V[k][p], vkq = V[k][q];
                    V[k][p] = cs * vkp - sn * vkq; V[k][q] = sn * vkp + cs * vkq;
                }
            }
    }
    int best = 0;
    for (int i = 1; i < TQ; ++i) if (A[i][i] > A[best][best]) best = i;
    T.mu = A[best][best];
    for (int i = 0; i < TQ; ++i) T.vec[i] = V[i][best] / sqrt(T.d[i]);
    double s = 0;
    for (int k = 0; k < TQ; ++k) s += T.d[k] * T.vec[k];
    T.at0 = s / T.mu;
}
}  // namespace

void ig_taper_eval(const double* eta, int n, double* psi) {
    std::call_once(g_taper_once, build_taper);
    const Taper& T = g_taper;
    for (int i = 0; i < n; ++i) {
        double e = eta[i];
        if (!(fabs(e) < 1.0)) { psi[i] = 0.0; continue; }
        double s = 0;
        for (int k = 0; k < TQ; ++k) s += cos(TC * e * T.t[k]) * T.d[k] * T.vec[k];
        psi[i] = (s / T.mu) / T.at0;
    }
}

// ---------------------------------------------------------------------------------------
__global__ void k_bank_twiddle(double2* __restrict__ W, int M) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= M) return;
    double s, c;
    sincospi(2.0 * (double)k / (double)M, &s, &c);
    W[k] = make_double2(c, -s);                       // exp(-j 2 pi k / M)
}

__global__ void k_bank_f(double2* __restrict__ f, const double* __restrict__ psi, int n, double du, double w) {
    int ai = blockIdx.x * blockDim.x + threadIdx.x, bi = blockIdx.y;
    if (ai >= n) return;
    double l = (double)(ai - n / 2) / ((double)n * du), m = (double)(bi - n / 2) / ((double)n * du);
    double r2 = l * l + m * m;
    double nm1 = sqrt(fmax(0.0, 1.0 - r2)) - 1.0;
    double s, c;
    sincos(2.0 * M_PI * w * nm1, &s, &c);
    double t = psi[ai] * psi[bi];
    f[(size_t)bi * n + ai] = make_double2(t * c, t * s);
}

// q(o,t) = (t-h)*beta - (o - shift): the oversampled sample that tap t reads at offset index o
__device__ __forceinline__ long long bank_q(int qi, int S, int beta, int shift) {
    int o = qi / S, t = qi - o * S;
    return (long long)(t - (S - 1) / 2) * beta - (o - shift);
}

__global__ void k_bank_g(double2* __restrict__ Gt, const double2* __restrict__ f, const double2* __restrict__ W,
                         int n, int M, int S, int beta, int shift) {
    const int Q = S * beta;
    int qi = blockIdx.x * blockDim.x + threadIdx.x, bi = blockIdx.y;
    if (qi >= Q) return;
    const long long q = bank_q(qi, S, beta, shift);
    long long ph = ((q * (long long)(-n / 2)) % M + M) % M;    // phase index of a = -n/2
    const long long step = ((q % M) + M) % M;
    double re = 0, im = 0;
    const double2* fr = f + (size_t)bi * n;
    for (int ai = 0; ai < n; ++ai) {
        double2 w = W[ph], x = fr[ai];
        re += x.x * w.x - x.y * w.y;
        im += x.x * w.y + x.y * w.x;
        ph += step; if (ph >= M) ph -= M;
    }
    Gt[(size_t)bi * Q + qi] = make_double2(re, im);
}

__global__ void k_bank_k(float2* __restrict__ K, const double2* __restrict__ Gt, const double2* __restrict__ W,
                         int n, int M, int S, int beta, int shift, double inv_a) {
    const int Q = S * beta;
    // output order [ov][ou][ty][tx]; thread = (ou, tx) flattened = qu index; block.y = (ov, ty) = qv index
    int qui = blockIdx.x * blockDim.x + threadIdx.x, qvi = blockIdx.y;
    if (qui >= Q) return;
    const long long q = bank_q(qvi, S, beta, shift);
    long long ph = ((q * (long long)(-n / 2)) % M + M) % M;
    const long long step = ((q % M) + M) % M;
    double re = 0, im = 0;
    for (int bi = 0; bi < n; ++bi) {
        double2 w = W[ph], x = Gt[(size_t)bi * Q + qui];
        re += x.x * w.x - x.y * w.y;
        im += x.x * w.y + x.y * w.x;
        ph += step; if (ph >= M) ph -= M;
    }
    const int ov = qvi / S, ty = qvi - ov * S, ou = qui / S, tx = qui - ou * S;
    K[(((size_t)ov * beta + ou) * S + ty) * S + tx] = make_float2((float)(re * inv_a), (float)(im * inv_a));
}

// zeta (eq 4.3 :1095): real part of the sum of each S x S matrix; one warp per matrix
__global__ void k_zeta(const float2* __restrict__ bank, const IgPlaneEntry* __restrict__ planes, int P, int b2,
                       double* __restrict__ zeta) {
    int m = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (m >= P * b2) return;
    int p = m / b2, tab = m - p * b2, S = planes[p].support;
    const float2* k = bank + planes[p].koff + (size_t)tab * S * S;
    double s = 0;
    for (int t = lane; t < S * S; t += 32) s += (double)k[t].x;
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) zeta[m] = s;
}

static int bank_inner_samples(int max_support) {
    int n = 1;
    while (n < 2 * max_support) n *= 2;
    return n;
}

size_t ig_bank_scratch_bytes(const ig_ctx* c) {
    size_t n = bank_inner_samples(c->max_support), M = n * c->prm.beta, Q = (size_t)c->max_support * c->prm.beta;
    return ig_align(n * 8) + ig_align(M * 16) + ig_align(n * n * 16) + ig_align(Q * n * 16);
}

int ig_launch_zeta(ig_ctx* c) {
    int b2 = c->prm.beta * c->prm.beta, m = c->prm.P * b2;
    k_zeta<<<(m * 32 + 255) / 256, 256, 0, c->stream>>>(c->d_bank, c->d_planes, c->prm.P, b2, c->d_zeta);
    IG_CUDA_OK(c, cudaGetLastError());
    return 1;
}

// ---------------------------------------------------------------------------------------
// Automatic support ("the pixel nearest to the edge with magnitude > 1e-3", reading 7):
// r_p = largest |q| (oversampled samples) on either axis through the centre with |C_p| > 1e-3 (C_0 peak = 1),
// searched over |q| <= beta*(max_support-1)/2; S_p = 2*ceil(r_p/beta) + 1. The axis profiles are 1-D DFTs of
// the column / row sums of f_p:  C_p[0][q] = sum_a (sum_b f[b][a]) W^(q a) / A.
__global__ void k_axis_sums(const double2* __restrict__ f, int n, double2* __restrict__ colsum, double2* __restrict__ rowsum) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double cr = 0, ci = 0, rr = 0, ri = 0;
    for (int k = 0; k < n; ++k) {
        double2 c = f[(size_t)k * n + i], r = f[(size_t)i * n + k];
        cr += c.x; ci += c.y; rr += r.x; ri += r.y;
    }
    colsum[i] = make_double2(cr, ci);
    rowsum[i] = make_double2(rr, ri);
}
__global__ void k_axis_radius(const double2* __restrict__ colsum, const double2* __restrict__ rowsum,
                              const double2* __restrict__ W, int n, int M, int qmax, double inv_a, double thr2,
                              int* __restrict__ radius) {
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > 2 * qmax) return;
    const long long q = t - qmax;
    long long ph = ((q * (long long)(-n / 2)) % M + M) % M;
    const long long step = ((q % M) + M) % M;
    double ur = 0, ui = 0, vr = 0, vi = 0;
    for (int a = 0; a < n; ++a) {
        const double2 w = W[ph], c = colsum[a], r = rowsum[a];
        ur += c.x * w.x - c.y * w.y; ui += c.x * w.y + c.y * w.x;
        vr += r.x * w.x - r.y * w.y; vi += r.x * w.y + r.y * w.x;
        ph += step; if (ph >= M) ph -= M;
    }
    ur *= inv_a; ui *= inv_a; vr *= inv_a; vi *= inv_a;
    const bool over = (ur * ur + ui * ui > thr2) || (vr * vr + vi * vi > thr2);
    if (over) atomicMax(radius, (int)(q < 0 ? -q : q));
}

// Fills table[P] (host) with the detected supports. Synchronises.
int ig_detect_supports(ig_ctx* c, char* scratch, size_t scratch_bytes, int* table) {
    if (scratch_bytes < ig_bank_scratch_bytes(c)) { c->err = "work buffer too small for the bank builder"; return -1; }
    const int n = bank_inner_samples(c->max_support), beta = c->prm.beta, M = n * beta, P = c->prm.P;
    double* d_psi = (double*)scratch;
    double2* d_W = (double2*)(scratch + ig_align((size_t)n * 8));
    double2* d_f = (double2*)((char*)d_W + ig_align((size_t)M * 16));
    char* g = (char*)d_f + ig_align((size_t)n * n * 16);          // the G area of the builder, free here
    double2* d_col = (double2*)g;
    double2* d_row = d_col + n;
    int* d_rad = (int*)(d_row + n);
    if ((size_t)n * 32 + (size_t)P * 4 > ig_align((size_t)c->max_support * beta * n * 16)) { c->err = "too many w-planes for the scratch area"; return -1; }
    std::vector<double> eta(n), psi(n);
    for (int i = 0; i < n; ++i) eta[i] = 2.0 * (double)(i - n / 2) / (double)n;
    ig_taper_eval(eta.data(), n, psi.data());
    double sum = 0;
    for (int i = 0; i < n; ++i) sum += psi[i];
    const double inv_a = 1.0 / (sum * sum);
    IG_CUDA_OK(c, cudaMemcpyAsync(d_psi, psi.data(), (size_t)n * 8, cudaMemcpyHostToDevice, c->stream));
    IG_CUDA_OK(c, cudaMemsetAsync(d_rad, 0, (size_t)P * 4, c->stream));
    IG_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    k_bank_twiddle<<<(M + 255) / 256, 256, 0, c->stream>>>(d_W, M);
    const int qmax = beta * ((c->max_support - 1) / 2);
    for (int p = 0; p < P; ++p) {
        const double w = P == 1 ? 0.0 : c->w_max * ((double)p / (P - 1)) * ((double)p / (P - 1));
        k_bank_f<<<dim3((n + 127) / 128, n), 128, 0, c->stream>>>(d_f, d_psi, n, c->du, w);
        k_axis_sums<<<(n + 127) / 128, 128, 0, c->stream>>>(d_f, n, d_col, d_row);
        k_axis_radius<<<(2 * qmax + 1 + 127) / 128, 128, 0, c->stream>>>(d_col, d_row, d_W, n, M, qmax, inv_a, 1e-3 * 1e-3, d_rad + p);
    }
    IG_CUDA_OK(c, cudaGetLastError());
    std::vector<int> rad(P);
    IG_CUDA_OK(c, cudaMemcpyAsync(rad.data(), d_rad, (size_t)P * 4, cudaMemcpyDeviceToHost, c->stream));
    IG_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    for (int p = 0; p < P; ++p) {
        int S = 2 * ((rad[p] + beta - 1) / beta) + 1;
        table[p] = S > c->max_support ? c->max_support : S;
    }
    return 3 * P + 1;
}

int ig_launch_bank(ig_ctx* c, char* scratch, size_t scratch_bytes) {
    if (scratch_bytes < ig_bank_scratch_bytes(c)) { c->err = "work buffer too small for the bank builder"; return -1; }
    const int n = bank_inner_samples(c->max_support), beta = c->prm.beta, M = n * beta;
    double* d_psi = (double*)scratch;
    double2* d_W = (double2*)(scratch + ig_align((size_t)n * 8));
    double2* d_f = (double2*)((char*)d_W + ig_align((size_t)M * 16));
    double2* d_G = (double2*)((char*)d_f + ig_align((size_t)n * n * 16));
    std::vector<double> eta(n), psi(n);
    for (int i = 0; i < n; ++i) eta[i] = 2.0 * (double)(i - n / 2) / (double)n;
    ig_taper_eval(eta.data(), n, psi.data());
    double sum = 0;
    for (int i = 0; i < n; ++i) sum += psi[i];
    const double inv_a = 1.0 / (sum * sum);
    IG_CUDA_OK(c, cudaMemcpyAsync(d_psi, psi.data(), (size_t)n * 8, cudaMemcpyHostToDevice, c->stream));
    IG_CUDA_OK(c, cudaStreamSynchronize(c->stream));   // psi is a stack-lifetime host buffer
    int launches = 0;
    k_bank_twiddle<<<(M + 255) / 256, 256, 0, c->stream>>>(d_W, M);
    ++launches;
    for (int p = 0; p < c->prm.P; ++p) {
        const int S = c->support[p], Q = S * beta;
        const double w = c->prm.P == 1 ? 0.0 : c->w_max * ((double)p / (c->prm.P - 1)) * ((double)p / (c->prm.P - 1));
        k_bank_f<<<dim3((n + 127) / 128, n), 128, 0, c->stream>>>(d_f, d_psi, n, c->du, w);
        k_bank_g<<<dim3((Q + 127) / 128, n), 128, 0, c->stream>>>(d_G, d_f, d_W, n, M, S, beta, c->prm.shift);
        k_bank_k<<<dim3((Q + 127) / 128, Q), 128, 0, c->stream>>>(c->d_bank + c->koff[p], d_G, d_W, n, M, S, beta,
                                                                  c->prm.shift, inv_a);
        launches += 3;
    }
    IG_CUDA_OK(c, cudaGetLastError());
    int z = ig_launch_zeta(c);
    if (z < 0) return -1;
    return launches + z;
}
