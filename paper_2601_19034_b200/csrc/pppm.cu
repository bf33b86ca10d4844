// pppm.cu -- steps a7P-1..5 of SURVEY.md 8(a): PPPM evaluation of the reciprocal-space part
// (PAPER.md II.F, Eq. 34-38; readings G2, S10, S11):
//   1. charge assignment with the order-5 cardinal B-spline (Eq. 35)
//   2. forward 3-D FFT of the charge mesh (hand-written, shared memory, no cuFFT; :302)
//   3. multiply by the optimised influence function G^opt (Eq. 36), energy (Eq. 34) and virial (Eq. 22)
//   4. inverse 3-D FFTs.  The four real fields F^-1[S G], F^-1[i k_a S G] (Eq. 37, 38; "3 + 1 backward
//      FFTs", :302) are packed pairwise into TWO complex transforms: M1 = Phi + i E_x, M2 = E_y + i E_z.
//   5. back-interpolation of phi^k_i and F^{k,static}_i with the same B-spline.
//
// FFT: one block transforms a tile of B = 16 lines held in shared memory as sm[k][b] (b fastest, so
// every butterfly access is a contiguous 128-byte row segment: conflict-free for any stride).  In-place
// decimation-in-frequency, radix 4 (+ one radix-2 stage when log2 n is odd); the digit-reversed order
// is undone for free when the rows are written back.  Strided axes move 128-byte row segments, the
// contiguous axis moves whole lines, so global traffic is coalesced in all three passes.
#include "qnep_internal.cuh"

#include <cmath>

namespace {

constexpr int FFT_B = 16;          // lines per tile
constexpr int FFT_BP = FFT_B + 1;  // padded row
constexpr int FFT_MAXN = 512;

__device__ __forceinline__ void bspline5(float dx, float* __restrict__ w)
{
    // centred cardinal B-spline of order 5 on mesh offsets -2..2 (reading S10)
    const float d2 = dx * dx, d3 = d2 * dx, d4 = d2 * d2;
    w[0] = (1.f - 8.f * dx + 24.f * d2 - 32.f * d3 + 16.f * d4) * (1.f / 384.f);
    w[1] = (19.f - 44.f * dx + 24.f * d2 + 16.f * d3 - 16.f * d4) * (1.f / 96.f);
    w[2] = (115.f - 120.f * d2 + 48.f * d4) * (1.f / 192.f);
    w[3] = (19.f + 44.f * dx + 24.f * d2 - 16.f * d3 - 16.f * d4) * (1.f / 96.f);
    w[4] = (1.f + 8.f * dx + 24.f * d2 + 32.f * d3 + 16.f * d4) * (1.f / 384.f);
}

__device__ __forceinline__ void stencil_indices(int packed, const int* grid, int (*idx)[5])
{
    const int m[3] = {packed & 1023, (packed >> 10) & 1023, (packed >> 20) & 1023};
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int o = 0; o < 5; ++o) {
            int v = m[a] + o - 2;
            v = v < 0 ? v + grid[a] : (v >= grid[a] ? v - grid[a] : v);
            idx[a][o] = v;
        }
}

// ---- 1. spreading ------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
k_spread(int64_t N, Geometry g, const float4* __restrict__ mfrac, const int* __restrict__ mi0,
         const float* __restrict__ q, float* __restrict__ mesh)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const float4 fr = mfrac[p];
    float wx[5], wy[5], wz[5];
    bspline5(fr.x, wx); bspline5(fr.y, wy); bspline5(fr.z, wz);
    int idx[3][5];
    stencil_indices(mi0[p], g.grid, idx);
    const float qi = q[p];
#pragma unroll
    for (int a = 0; a < 5; ++a) {
        const float qa = qi * wx[a];
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const float qab = qa * wy[b];
            float* row = mesh + ((int64_t)idx[0][a] * g.grid[1] + idx[1][b]) * g.grid[2];
#pragma unroll
            for (int c = 0; c < 5; ++c) atomicAdd(row + idx[2][c], qab * wz[c]);
        }
    }
}

// ---- 2./4. FFT along one axis -----------------------------------------------------------------
struct FftPlan {
    int n, log2n;
    int axis;                 // 0, 1, 2 of an [n0][n1][n2] array (n2 fastest)
    int n0, n1, n2;
    int sign;                 // -1 forward, +1 inverse (both unnormalised; reading S11)
};

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

template <bool IN_REAL>
__global__ void __launch_bounds__(256)
k_fft_axis(FftPlan pl, const float* __restrict__ in_real, const float2* in, float2* out,   // in may alias out (in place)
           const float2* __restrict__ twiddle /* [n] e^{-2 pi i t / n} */, const int* __restrict__ perm /* pos -> freq */)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* sm = reinterpret_cast<float2*>(smem_raw);                 // [n][FFT_BP]
    float2* tw = sm + (size_t)pl.n * FFT_BP;                          // [n]
    int* pm = reinterpret_cast<int*>(tw + pl.n);                      // [n]
    const int n = pl.n;
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int t = tid; t < n; t += nt) {
        float2 w = twiddle[t];
        if (pl.sign > 0) w.y = -w.y;
        tw[t] = w;
        pm[t] = perm[t];
    }
    // tile addressing
    int64_t base;          // element offset of (k = 0, b = 0)
    int64_t stride_k;      // between consecutive k of one line
    const int64_t tile = blockIdx.x;
    if (pl.axis == 2) { base = tile * FFT_B * (int64_t)n; stride_k = 1; }
    else if (pl.axis == 1) {
        const int tiles_per_plane = pl.n2 / FFT_B;
        base = (tile / tiles_per_plane) * (int64_t)pl.n1 * pl.n2 + (tile % tiles_per_plane) * FFT_B;
        stride_k = pl.n2;
    } else { base = tile * FFT_B; stride_k = (int64_t)pl.n1 * pl.n2; }
    // load
    if (pl.axis == 2) {
        for (int e = tid; e < n * FFT_B; e += nt) {
            const int b = e / n, k = e - b * n;
            float2 v;
            if (IN_REAL) v = make_float2(in_real[base + e], 0.f);
            else v = in[base + e];
            sm[k * FFT_BP + b] = v;
        }
    } else {
        for (int e = tid; e < n * FFT_B; e += nt) {
            const int k = e / FFT_B, b = e - k * FFT_B;
            sm[k * FFT_BP + b] = in[base + k * stride_k + b];
        }
    }
    __syncthreads();
    // DIF stages
    int m = n;                                  // current sub-transform length
    while (m >= 4) {
        const int qn = m >> 2;                  // quarter
        const int tstep = n / m;                // twiddle index step
        for (int e = tid; e < (n >> 2) * FFT_B; e += nt) {
            const int b = e % FFT_B;
            const int bf = e / FFT_B;           // butterfly id 0..n/4-1
            const int j = bf % qn;
            const int blk = bf / qn;
            const int i0 = blk * m + j;
            float2* p0 = sm + (i0)*FFT_BP + b;
            float2* p1 = p0 + qn * FFT_BP;
            float2* p2 = p1 + qn * FFT_BP;
            float2* p3 = p2 + qn * FFT_BP;
            const float2 a0 = *p0, a1 = *p1, a2 = *p2, a3 = *p3;
            const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), d13 = csub(a1, a3);
            // omega * d13, omega = -i (forward) or +i (inverse)
            const float2 t3 = pl.sign < 0 ? make_float2(d13.y, -d13.x) : make_float2(-d13.y, d13.x);
            const float2 y0 = cadd(t0, t2), y1 = cadd(t1, t3), y2 = csub(t0, t2), y3 = csub(t1, t3);
            const int ti = j * tstep;
            *p0 = y0;
            *p1 = cmul(y1, tw[ti]);
            *p2 = cmul(y2, tw[2 * ti]);
            *p3 = cmul(y3, tw[3 * ti]);
        }
        __syncthreads();
        m >>= 2;
    }
    if (m == 2) {
        for (int e = tid; e < (n >> 1) * FFT_B; e += nt) {
            const int b = e % FFT_B;
            const int blk = e / FFT_B;
            float2* p0 = sm + (2 * blk) * FFT_BP + b;
            float2* p1 = p0 + FFT_BP;
            const float2 a0 = *p0, a1 = *p1;
            *p0 = cadd(a0, a1);
            *p1 = csub(a0, a1);
        }
        __syncthreads();
    }
    // store: row `pos` holds frequency pm[pos]
    if (pl.axis == 2) {
        for (int e = tid; e < n * FFT_B; e += nt) {
            const int b = e / n, pos = e - b * n;
            out[base + (int64_t)b * n + pm[pos]] = sm[pos * FFT_BP + b];
        }
    } else {
        for (int e = tid; e < n * FFT_B; e += nt) {
            const int pos = e / FFT_B, b = e - pos * FFT_B;
            out[base + pm[pos] * stride_k + b] = sm[pos * FFT_BP + b];
        }
    }
}

// ---- 3. influence function ----------------------------------------------------------------------
// tables per axis a (offset a * FFT_MAXN): A[m] = exp(-k^2/4 alpha^2) sinc^10(pi n/N) / d(z)^2, kk[m] = k (true, for
// k^2), kd[m] = k with the Nyquist entry zeroed (for the i k multiplier, S11).
__global__ void __launch_bounds__(256)
k_influence(Geometry g, const float* __restrict__ tabA, const float* __restrict__ tabK, const float* __restrict__ tabKd,
            double c0 /* 2 pi / Omega */, double inv4a2, const float2* S, float2* M1,   // S may alias M1
            float2* __restrict__ M2, double* __restrict__ sums)
{
    __shared__ double sh_red[32];
    const int64_t ng = (int64_t)g.grid[0] * g.grid[1] * g.grid[2];
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int64_t m = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; m < ng; m += (int64_t)gridDim.x * blockDim.x) {
        const int m2 = (int)(m % g.grid[2]);
        const int m1 = (int)((m / g.grid[2]) % g.grid[1]);
        const int m0 = (int)(m / ((int64_t)g.grid[2] * g.grid[1]));
        const float kx = tabK[m0], ky = tabK[FFT_MAXN + m1], kz = tabK[2 * FFT_MAXN + m2];
        const float k2 = kx * kx + ky * ky + kz * kz;
        float2 phi = make_float2(0.f, 0.f);
        const float2 s = S[m];
        if (k2 > 0.f) {
            const float G = (float)c0 * tabA[m0] * tabA[FFT_MAXN + m1] * tabA[2 * FFT_MAXN + m2] / k2;
            phi = make_float2(G * s.x, G * s.y);
            const double e = QNEP_K_COULOMB * (double)G * ((double)s.x * s.x + (double)s.y * s.y);
            const double bf = 2.0 * inv4a2 + 2.0 / (double)k2;
            acc[0] += e;
            acc[1] += e * (1.0 - bf * kx * kx);
            acc[2] += e * (-bf * kx * ky);
            acc[3] += e * (-bf * kx * kz);
            acc[4] += e * (1.0 - bf * ky * ky);
            acc[5] += e * (-bf * ky * kz);
            acc[6] += e * (1.0 - bf * kz * kz);
        }
        const float kdx = tabKd[m0], kdy = tabKd[FFT_MAXN + m1], kdz = tabKd[2 * FFT_MAXN + m2];
        // M1 = Phi + i (i kx Phi) = (1 - kx) Phi ;  M2 = i ky Phi + i (i kz Phi) = (-kz + i ky) Phi
        M1[m] = make_float2((1.f - kdx) * phi.x, (1.f - kdx) * phi.y);
        M2[m] = make_float2(-kdz * phi.x - kdy * phi.y, -kdz * phi.y + kdy * phi.x);
    }
    const int slot[7] = {SUM_U_K, SUM_W0 + 0, SUM_W0 + 1, SUM_W0 + 2, SUM_W0 + 4, SUM_W0 + 5, SUM_W0 + 8};
    const int mirror[7] = {-1, -1, SUM_W0 + 3, SUM_W0 + 6, -1, SUM_W0 + 7, -1};
#pragma unroll
    for (int a = 0; a < 7; ++a) {
        double v = acc[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) sh_red[threadIdx.x >> 5] = v;
        __syncthreads();
        if (threadIdx.x < 32) {
            double r = threadIdx.x < (blockDim.x >> 5) ? sh_red[threadIdx.x] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
            if (threadIdx.x == 0) {
                atomicAdd(&sums[slot[a]], r);
                if (mirror[a] >= 0) atomicAdd(&sums[mirror[a]], r);
            }
        }
    }
}

// ---- 5. back-interpolation ------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
k_gather(int64_t N, Geometry g, const float4* __restrict__ mfrac, const int* __restrict__ mi0,
         const float* __restrict__ q, const float2* __restrict__ M1, const float2* __restrict__ M2, int add_to_Fs,
         float* __restrict__ phik, float* __restrict__ Fs)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const float4 fr = mfrac[p];
    float wx[5], wy[5], wz[5];
    bspline5(fr.x, wx); bspline5(fr.y, wy); bspline5(fr.z, wz);
    int idx[3][5];
    stencil_indices(mi0[p], g.grid, idx);
    float ph = 0.f, ex = 0.f, ey = 0.f, ez = 0.f;
#pragma unroll
    for (int a = 0; a < 5; ++a) {
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const float wab = wx[a] * wy[b];
            const int64_t row = ((int64_t)idx[0][a] * g.grid[1] + idx[1][b]) * g.grid[2];
#pragma unroll
            for (int c = 0; c < 5; ++c) {
                const float w = wab * wz[c];
                const float2 u = M1[row + idx[2][c]];
                const float2 v = M2[row + idx[2][c]];
                ph = fmaf(w, u.x, ph); ex = fmaf(w, u.y, ex);
                ey = fmaf(w, v.x, ey); ez = fmaf(w, v.y, ez);
            }
        }
    }
    const float c2k = 2.f * (float)QNEP_K_COULOMB;
    phik[p] = c2k * ph;                                   // bracket of Eq. 38
    const float cq = -c2k * q[p];                         // Eq. 37
    if (add_to_Fs) { Fs[p] += cq * ex; Fs[N + p] += cq * ey; Fs[2 * N + p] += cq * ez; }
    else { Fs[p] = cq * ex; Fs[N + p] = cq * ey; Fs[2 * N + p] = cq * ez; }
}

int launch_fft3d(qnep_handle* h, const float* in_real, float2* data, int sign, cudaStream_t s)
{
    const int n0 = h->geo.grid[0], n1 = h->geo.grid[1], n2 = h->geo.grid[2];
    const int order_fwd[3] = {2, 1, 0}, order_inv[3] = {0, 1, 2};
    for (int step = 0; step < 3; ++step) {
        const int axis = sign < 0 ? order_fwd[step] : order_inv[step];
        const int n = axis == 0 ? n0 : (axis == 1 ? n1 : n2);
        FftPlan pl;
        pl.n = n; pl.log2n = 0; while ((1 << pl.log2n) < n) ++pl.log2n;
        pl.axis = axis; pl.n0 = n0; pl.n1 = n1; pl.n2 = n2; pl.sign = sign;
        const int64_t lines = (int64_t)n0 * n1 * n2 / n;
        const int tiles = (int)(lines / FFT_B);
        const size_t smem = sizeof(float2) * ((size_t)n * FFT_BP + n) + sizeof(int) * n;
        const int threads = std::min(256, std::max(32, n * FFT_B / 4));
        const bool real_in = (in_real != nullptr) && step == 0 && sign < 0;
        if (real_in)
            k_fft_axis<true><<<tiles, threads, smem, s>>>(pl, in_real, nullptr, data, h->d_twiddle + axis * FFT_MAXN,
                                                          reinterpret_cast<const int*>(h->d_twiddle + 3 * FFT_MAXN) + axis * FFT_MAXN);
        else
            k_fft_axis<false><<<tiles, threads, smem, s>>>(pl, nullptr, data, data, h->d_twiddle + axis * FFT_MAXN,
                                                           reinterpret_cast<const int*>(h->d_twiddle + 3 * FFT_MAXN) + axis * FFT_MAXN);
        h->launches += 1;
    }
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

double alias_den(double z)
{
    const double z2 = z * z;   // Eq. 36 denominator polynomial (reading G2: -17/189)
    return 1.0 - 5.0 / 3.0 * z2 + 7.0 / 9.0 * z2 * z2 - 17.0 / 189.0 * z2 * z2 * z2 + 2.0 / 2835.0 * z2 * z2 * z2 * z2;
}

}  // namespace

// tables: twiddles, digit-reversal permutations and the separable factors of G^opt (Eq. 36)
int qnep_setup_pppm(qnep_handle* h)
{
    const int* grid = h->es.grid;
    for (int a = 0; a < 3; ++a) {
        const int n = grid[a];
        if (n < FFT_B || n > FFT_MAXN || (n & (n - 1))) { h->err = "PPPM grid must be a power of two in 16..512"; return QNEP_ERR_UNSUPPORTED; }
    }
    if (h->es.order != 5) { h->err = "PPPM order must be 5"; return QNEP_ERR_UNSUPPORTED; }
    const int64_t ng = (int64_t)grid[0] * grid[1] * grid[2];
    if (ng != h->ngrid) {
        cudaFree(h->d_mesh); cudaFree(h->d_cm1); cudaFree(h->d_cm2);
        h->d_mesh = nullptr; h->d_cm1 = nullptr; h->d_cm2 = nullptr;
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_mesh, sizeof(float) * ng));
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_cm1, sizeof(float2) * ng));
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_cm2, sizeof(float2) * ng));
        h->ngrid = ng;
    }
    if (!h->d_twiddle) QNEP_CUDA_OK(h, cudaMalloc(&h->d_twiddle, sizeof(float2) * 3 * FFT_MAXN + sizeof(int) * 3 * FFT_MAXN));
    if (!h->d_gtab) QNEP_CUDA_OK(h, cudaMalloc(&h->d_gtab, sizeof(float) * 9 * FFT_MAXN));
    std::vector<float2> tw(3 * FFT_MAXN, make_float2(0.f, 0.f));
    std::vector<int> pm(3 * FFT_MAXN, 0);
    std::vector<float> tab(9 * FFT_MAXN, 0.f);
    const double L[3] = {h->box[0], h->box[4], h->box[8]};
    for (int a = 0; a < 3; ++a) {
        const int n = grid[a];
        for (int t = 0; t < n; ++t) {
            const double ang = -2.0 * M_PI * t / n;
            tw[a * FFT_MAXN + t] = make_float2((float)cos(ang), (float)sin(ang));
        }
        // position -> frequency after the DIF stages: pos = sum_i c_i q_i, freq = c_1 + r_1 (c_2 + r_2 (...))
        for (int pos = 0; pos < n; ++pos) {
            int rem = pos, m = n, freq = 0, weight = 1;
            while (m >= 4) { const int q = m / 4; const int c = rem / q; rem -= c * q; freq += c * weight; weight *= 4; m = q; }
            if (m == 2) { const int c = rem; freq += c * weight; }
            pm[a * FFT_MAXN + pos] = freq;
        }
        for (int m = 0; m < n; ++m) {
            const int nn = m < n / 2 ? m : m - n;                 // -N/2 <= n < N/2 (:285)
            const double k = 2.0 * M_PI * nn / L[a];
            const double x = M_PI * nn / n;
            const double sc = x == 0.0 ? 1.0 : sin(x) / x;
            const double d = alias_den(sin(x));
            tab[a * FFT_MAXN + m] = (float)(exp(-k * k / (4.0 * h->alpha * h->alpha)) * pow(sc, 10) / (d * d));
            tab[(3 + a) * FFT_MAXN + m] = (float)k;
            tab[(6 + a) * FFT_MAXN + m] = (2 * nn == -n) ? 0.f : (float)k;
        }
    }
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_twiddle, tw.data(), sizeof(float2) * 3 * FFT_MAXN, cudaMemcpyHostToDevice));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_twiddle + 3 * FFT_MAXN, pm.data(), sizeof(int) * 3 * FFT_MAXN, cudaMemcpyHostToDevice));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_gtab, tab.data(), sizeof(float) * 9 * FFT_MAXN, cudaMemcpyHostToDevice));
    static bool attr = false;
    if (!attr) {
        QNEP_CUDA_OK(h, cudaFuncSetAttribute(k_fft_axis<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
        QNEP_CUDA_OK(h, cudaFuncSetAttribute(k_fft_axis<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024));
        attr = true;
    }
    return QNEP_OK;
}

int qnep_launch_pppm(qnep_handle* h, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 127) / 128);
    const double L[3] = {h->box[0], h->box[4], h->box[8]};
    QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_mesh, 0, sizeof(float) * h->ngrid, s));
    k_spread<<<nb, 128, 0, s>>>(N, h->geo, h->d_mfrac, h->d_mi0, h->d_q, h->d_mesh);
    h->launches += 1;
    int rc = launch_fft3d(h, h->d_mesh, h->d_cm1, -1, s);
    if (rc) return rc;
    const int nblk = (int)std::min<int64_t>((h->ngrid + 255) / 256, 148 * 8);
    k_influence<<<nblk, 256, 0, s>>>(h->geo, h->d_gtab, h->d_gtab + 3 * FFT_MAXN, h->d_gtab + 6 * FFT_MAXN,
                                     2.0 * M_PI / (L[0] * L[1] * L[2]), 1.0 / (4.0 * h->alpha * h->alpha), h->d_cm1,
                                     h->d_cm1, h->d_cm2, h->d_sums);
    h->launches += 1;
    rc = launch_fft3d(h, nullptr, h->d_cm1, +1, s);
    if (rc) return rc;
    rc = launch_fft3d(h, nullptr, h->d_cm2, +1, s);
    if (rc) return rc;
    k_gather<<<nb, 128, 0, s>>>(N, h->geo, h->d_mfrac, h->d_mi0, h->d_q, h->d_cm1, h->d_cm2, h->model.mode == 1 ? 1 : 0,
                                h->d_phik, h->d_Fs);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}
