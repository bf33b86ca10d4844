// electro.cu -- steps a6, a7E, a8, a9 of SURVEY.md 8(a):
//   real-space Ewald term (Eq. 6, 15, 16; truncated at rc_r as the paper defines, :89),
//   self term (Eq. 10, 23), direct Ewald summation of the reciprocal part (Eq. 7-9, 18, 19, 21-22)
//   and the assembly of phi_i = dU^ES/dq_i with its mean (reading S6).
#include "qnep_internal.cuh"

#include <cmath>

namespace {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ double block_sum(double v, double* sh)
{
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = lane < (blockDim.x >> 5) ? sh[lane] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

// ---- a6: real-space term over the live radial list of this step (mode 1) ---------------------
__global__ void __launch_bounds__(128)
k_realspace(int64_t N, Geometry g, const float4* __restrict__ xyzt, const int4* __restrict__ nl, int cap,
            const int* __restrict__ nn, const float* __restrict__ q, float alpha, float* __restrict__ phir,
            float* __restrict__ Fs, double* __restrict__ sums, float* __restrict__ Wat /* [9][N] or null */)
{
    __shared__ double sh_red[32];
    const CellVecs cv = qnep_cell_vecs(g.cellv, g.triclinic);
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const float Kc = (float)QNEP_K_COULOMB;
    const float two_a_sqrtpi = 2.f * alpha * 0.5641895835477563f;
    float W[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    float Ur = 0.f;
    if (p < N) {
        const float4 xi = xyzt[p];
        const float qi = q[p];
        float phi = 0.f, Fx = 0.f, Fy = 0.f, Fz = 0.f;
        const int n = nn[p];
        const int* words = reinterpret_cast<const int*>(nl + qnep_tiled_base(p, cap / 4));   // slot s: int4 s / 4, lane s % 4
        for (int s = 0; s < n; ++s) {
            const int e = words[(int64_t)(s >> 2) * (4 * QNEP_TILE) + (s & 3)];
            const int j = e & QNEP_NL_MASK;
            const float4 xj = xyzt[j];
            float dx = xj.x - xi.x, dy = xj.y - xi.y, dz = xj.z - xi.z;
            qnep_add_image_shift(e, cv, dx, dy, dz);
            const float r2 = dx * dx + dy * dy + dz * dz;
            if (r2 >= g.rc_r2) continue;
            const float r = sqrtf(r2), rinv = 1.f / r;
            const float qj = q[j];
            const float ar = alpha * r;
            const float ec = erfcf(ar);
            const float e1 = ec * rinv;                                   // erfc(a r) / r
            phi = fmaf(qj, e1, phi);
            // [2 a r exp(-a^2 r^2)/sqrt(pi) + erfc(a r)] / r^3
            const float br = (two_a_sqrtpi * r * __expf(-ar * ar) + ec) * rinv * rinv * rinv;
            const float w = qi * qj * br;
            Fx = fmaf(-w, dx, Fx); Fy = fmaf(-w, dy, Fy); Fz = fmaf(-w, dz, Fz);
            W[0] = fmaf(w * dx, dx, W[0]); W[1] = fmaf(w * dx, dy, W[1]); W[2] = fmaf(w * dx, dz, W[2]);
            W[3] = fmaf(w * dy, dy, W[3]); W[4] = fmaf(w * dy, dz, W[4]); W[5] = fmaf(w * dz, dz, W[5]);
        }
        phir[p] = Kc * phi;
        Fs[p] = Kc * Fx; Fs[N + p] = Kc * Fy; Fs[2 * N + p] = Kc * Fz;
        Ur = 0.5f * Kc * qi * phi;
        if (Wat) {
            // per-atom virial of the real-space static part: W_i = sum_j r_ij (x) F_ji (Eq. 12 with Eq. 15)
            const float h = 0.5f * Kc;
            Wat[p] = h * W[0]; Wat[N + p] = h * W[1]; Wat[2 * N + p] = h * W[2];
            Wat[3 * N + p] = h * W[1]; Wat[4 * N + p] = h * W[3]; Wat[5 * N + p] = h * W[4];
            Wat[6 * N + p] = h * W[2]; Wat[7 * N + p] = h * W[4]; Wat[8 * N + p] = h * W[5];
        }
    }
    const double u = block_sum((double)Ur, sh_red);
    if (threadIdx.x == 0) atomicAdd(&sums[SUM_U_R], u);
    const int map[6][2] = {{0, 0}, {0, 1}, {0, 2}, {1, 1}, {1, 2}, {2, 2}};
#pragma unroll
    for (int a = 0; a < 6; ++a) {
        const double w = block_sum(0.5 * (double)Kc * (double)W[a], sh_red);
        if (threadIdx.x == 0) {
            atomicAdd(&sums[SUM_W0 + 3 * map[a][0] + map[a][1]], w);
            if (map[a][0] != map[a][1]) atomicAdd(&sums[SUM_W0 + 3 * map[a][1] + map[a][0]], w);
        }
    }
}

// ---- a8 + a9: phi = phi^k + phi^r + phi^s, sum of phi, U^s ------------------------------------
__global__ void k_phi_finalize(int64_t N, int mode, int have_k, float alpha, const float* __restrict__ q,
                               const float* __restrict__ phik, const float* __restrict__ phir, float* __restrict__ phi,
                               double* __restrict__ sums)
{
    __shared__ double sh_red[32];
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double ph = 0.0, us = 0.0;
    if (p < N) {
        float v = have_k ? phik[p] : 0.f;
        if (mode == 1 && have_k) {
            const double qi = q[p];
            const double c = QNEP_K_COULOMB * (double)alpha * 0.5641895835477563;   // K alpha / sqrt(pi)
            us = -c * qi * qi;                                                      // Eq. 10
            v += phir[p] + (float)(-2.0 * c * qi);                                  // Eq. 16 bracket + Eq. 23
        }
        phi[p] = v;
        ph = v;
    }
    const double s1 = block_sum(ph, sh_red);
    const double s2 = block_sum(us, sh_red);
    if (threadIdx.x == 0) { atomicAdd(&sums[SUM_PHI], s1); if (mode == 1) atomicAdd(&sums[SUM_U_S], s2); }
}

// ---- a7E: direct Ewald sum -------------------------------------------------------------------
// e^{i 2 pi n f_a} for n = 0..nmax, per atom and axis (f = fractional coordinate, computed in fp64)
__global__ void k_ewald_phases(int64_t N, const double* __restrict__ pos, const int* __restrict__ sidx, Geometry g,
                               int nmax, float2* __restrict__ eph)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int i = sidx[p];
    const double r[3] = {pos[i], pos[N + i], pos[2 * N + i]};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double f = r[0] * g.hinv[a] + r[1] * g.hinv[3 + a] + r[2] * g.hinv[6 + a];
        f -= floor(f);
        for (int n = 0; n <= nmax; ++n) {
            double t = 2.0 * n * f;
            t -= 2.0 * floor(0.5 * t);                       // reduce to [0, 2)
            float sn, cs;
            sincospif((float)t, &sn, &cs);
            eph[((int64_t)a * (nmax + 1) + n) * N + p] = make_float2(cs, sn);
        }
    }
}

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

__device__ __forceinline__ float2 phase_of(const float2* __restrict__ eph, int64_t N, int nmax, int64_t p, int kint)
{
    const int n0 = (kint & 1023) - 512, n1 = ((kint >> 10) & 1023) - 512, n2 = ((kint >> 20) & 1023) - 512;
    float2 e0 = eph[((int64_t)0 * (nmax + 1) + abs(n0)) * N + p];
    float2 e1 = eph[((int64_t)1 * (nmax + 1) + abs(n1)) * N + p];
    float2 e2 = eph[((int64_t)2 * (nmax + 1) + abs(n2)) * N + p];
    if (n0 < 0) e0.y = -e0.y;
    if (n1 < 0) e1.y = -e1.y;
    if (n2 < 0) e2.y = -e2.y;
    return cmul(cmul(e0, e1), e2);                            // e^{+i k.r}
}

// S(k) = sum_i q_i e^{-i k.r_i}  (Eq. 8): one block per k
__global__ void __launch_bounds__(256)
k_ewald_sfac(int64_t N, int nmax, const float2* __restrict__ eph, const int* __restrict__ kint,
             const float* __restrict__ q, double2* __restrict__ S)
{
    __shared__ double sh_red[32];
    const int k = blockIdx.x;
    const int ki = kint[k];
    double sr = 0.0, si = 0.0;
    for (int64_t p = threadIdx.x; p < N; p += blockDim.x) {
        const float2 e = phase_of(eph, N, nmax, p, ki);
        const float qi = q[p];
        sr += (double)(qi * e.x);
        si -= (double)(qi * e.y);
    }
    const double a = block_sum(sr, sh_red);
    const double b = block_sum(si, sh_red);
    if (threadIdx.x == 0) S[k] = make_double2(a, b);
}

// U^k (Eq. 7) and W^k (Eq. 21-22) over the half sphere (factor 2 for -k)
__global__ void __launch_bounds__(256)
k_ewald_energy(int nk, const float4* __restrict__ kvec, const double2* __restrict__ S, double inv4a2,
               double* __restrict__ sums)
{
    __shared__ double sh_red[32];
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nk; k += gridDim.x * blockDim.x) {
        const float4 kv = kvec[k];
        const double2 s = S[k];
        const double e = 2.0 * QNEP_K_COULOMB * (double)kv.w * (s.x * s.x + s.y * s.y);
        const double k2 = (double)kv.x * kv.x + (double)kv.y * kv.y + (double)kv.z * kv.z;
        const double bf = 2.0 * inv4a2 + 2.0 / k2;
        acc[0] += e;
        acc[1] += e * (1.0 - bf * kv.x * kv.x);
        acc[2] += e * (-bf * kv.x * kv.y);
        acc[3] += e * (-bf * kv.x * kv.z);
        acc[4] += e * (1.0 - bf * kv.y * kv.y);
        acc[5] += e * (-bf * kv.y * kv.z);
        acc[6] += e * (1.0 - bf * kv.z * kv.z);
    }
    const int slot[7] = {SUM_U_K, SUM_W0 + 0, SUM_W0 + 1, SUM_W0 + 2, SUM_W0 + 4, SUM_W0 + 5, SUM_W0 + 8};
    const int mirror[7] = {-1, -1, SUM_W0 + 3, SUM_W0 + 6, -1, SUM_W0 + 7, -1};
#pragma unroll
    for (int a = 0; a < 7; ++a) {
        const double v = block_sum(acc[a], sh_red);
        if (threadIdx.x == 0) {
            atomicAdd(&sums[slot[a]], v);
            if (mirror[a] >= 0) atomicAdd(&sums[mirror[a]], v);
        }
    }
}

// phi^k_i = 2K sum_k G Re[S e^{ik.r_i}] (Eq. 19 bracket), F^k_i = 2K q_i sum_k k G Im[S e^{ik.r_i}] (Eq. 18)
template <bool ATOMV>
__global__ void __launch_bounds__(128)
k_ewald_atoms(int64_t N, int nk, int nmax, const float2* __restrict__ eph, const int* __restrict__ kint,
              const float4* __restrict__ kvec, const double2* __restrict__ S, const float* __restrict__ q, int add_to_Fs,
              float* __restrict__ phik, float* __restrict__ Fs, float inv4a2, int add_to_Wat, float* __restrict__ Wat)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    float phi = 0.f, fx = 0.f, fy = 0.f, fz = 0.f;
    float wv[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};           // xx, xy, xz, yy, yz, zz of sum_k G Re[S e^{ik.r}] B (Eq. 20-21)
    for (int k = 0; k < nk; ++k) {
        const float2 e = phase_of(eph, N, nmax, p, kint[k]);
        const float4 kv = kvec[k];
        const double2 sd = S[k];
        const float sr = (float)sd.x, si = (float)sd.y;
        const float re = sr * e.x - si * e.y;
        const float im = sr * e.y + si * e.x;
        phi = fmaf(kv.w, re, phi);
        const float gi = kv.w * im;
        fx = fmaf(gi, kv.x, fx); fy = fmaf(gi, kv.y, fy); fz = fmaf(gi, kv.z, fz);
        if (ATOMV) {
            const float gr = kv.w * re;
            const float k2 = kv.x * kv.x + kv.y * kv.y + kv.z * kv.z;
            const float bf = gr * (2.f * inv4a2 + 2.f / k2);
            wv[0] += gr - bf * kv.x * kv.x; wv[1] -= bf * kv.x * kv.y; wv[2] -= bf * kv.x * kv.z;
            wv[3] += gr - bf * kv.y * kv.y; wv[4] -= bf * kv.y * kv.z; wv[5] += gr - bf * kv.z * kv.z;
        }
    }
    const float c = 4.f * (float)QNEP_K_COULOMB;              // 2K, times 2 for the -k half
    phik[p] = c * phi;
    const float cq = c * q[p];
    if (add_to_Fs) { Fs[p] += cq * fx; Fs[N + p] += cq * fy; Fs[2 * N + p] += cq * fz; }
    else { Fs[p] = cq * fx; Fs[N + p] = cq * fy; Fs[2 * N + p] = cq * fz; }
    if (ATOMV) {
        // K q_i sum over the FULL sphere = 2 K q_i sum over the stored half
        const float cw = 2.f * (float)QNEP_K_COULOMB * q[p];
        const int row[9] = {0, 1, 2, 1, 3, 4, 2, 4, 5};
#pragma unroll
        for (int a = 0; a < 9; ++a) {
            const float v = cw * wv[row[a]];
            if (add_to_Wat) Wat[(int64_t)a * N + p] += v; else Wat[(int64_t)a * N + p] = v;
        }
    }
}

}  // namespace

int qnep_launch_realspace(qnep_handle* h, bool atomv, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 127) / 128);
    k_realspace<<<nb, 128, 0, s>>>(N, h->geo, h->d_xyzt, h->d_lvR, h->capLR, h->d_nlvR, h->d_q, (float)h->alpha, h->d_phir, h->d_Fs,
                                   h->d_sums, atomv ? h->d_Wat : nullptr);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int qnep_launch_phi_finalize(qnep_handle* h, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 255) / 256);
    k_phi_finalize<<<nb, 256, 0, s>>>(N, h->model.mode, h->es.method != 0 ? 1 : 0, (float)h->alpha, h->d_q, h->d_phik,
                                      h->d_phir, h->d_phi, h->d_sums);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

// k-vector list on the host (reading S7): half sphere, integer criterion n.n <= nmax2 when
// given, else |k| <= 2 pi alpha; G(k) of Eq. 9 in double, stored as float.
int qnep_setup_ewald(qnep_handle* h)
{
    const Geometry& g = h->geo;                          // any cell: k = 2 pi (n0 b*_0 + n1 b*_1 + n2 b*_2), b*_b = column b of h^-1 (:104)
    const double L[3] = {g.L[0], g.L[1], g.L[2]};        // lengths of the cell vectors (bound of the integer range, as in the oracle)
    const double vol = std::fabs(g.h[0] * (g.h[4] * g.h[8] - g.h[5] * g.h[7]) - g.h[1] * (g.h[3] * g.h[8] - g.h[5] * g.h[6]) +
                                 g.h[2] * (g.h[3] * g.h[7] - g.h[4] * g.h[6]));
    const double alpha = h->alpha;
    const double kmax = 2.0 * M_PI * alpha;
    int nmax[3];
    for (int a = 0; a < 3; ++a)
        nmax[a] = h->es.ewald_nmax2 > 0 ? (int)floor(sqrt((double)h->es.ewald_nmax2)) : (int)ceil(kmax * L[a] / (2.0 * M_PI)) + 1;
    int nm = std::max(nmax[0], std::max(nmax[1], nmax[2]));
    if (nm > 500) { h->err = "Ewald k-range too large"; return QNEP_ERR_UNSUPPORTED; }
    std::vector<float4> kv;
    std::vector<int> ki;
    for (int n0 = 0; n0 <= nmax[0]; ++n0)
        for (int n1 = -nmax[1]; n1 <= nmax[1]; ++n1)
            for (int n2 = -nmax[2]; n2 <= nmax[2]; ++n2) {
                const bool half = n0 > 0 || (n0 == 0 && (n1 > 0 || (n1 == 0 && n2 > 0)));
                if (!half) continue;
                double k[3];
                for (int a = 0; a < 3; ++a) k[a] = 2.0 * M_PI * (n0 * g.hinv[3 * a] + n1 * g.hinv[3 * a + 1] + n2 * g.hinv[3 * a + 2]);
                const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                if (h->es.ewald_nmax2 > 0) { if (n0 * n0 + n1 * n1 + n2 * n2 > h->es.ewald_nmax2) continue; }
                else if (k2 > kmax * kmax * (1.0 + 1e-12)) continue;
                const double G = 2.0 * M_PI / vol * exp(-k2 / (4.0 * alpha * alpha)) / k2;
                kv.push_back(make_float4((float)k[0], (float)k[1], (float)k[2], (float)G));
                ki.push_back((n0 + 512) | ((n1 + 512) << 10) | ((n2 + 512) << 20));
            }
    cudaFree(h->d_kvec); cudaFree(h->d_kint); cudaFree(h->d_S); cudaFree(h->d_ephase);
    h->d_kvec = nullptr; h->d_kint = nullptr; h->d_S = nullptr; h->d_ephase = nullptr;
    h->nk = (int)kv.size();
    h->ew_nmax = nm;
    if (h->nk == 0) return QNEP_OK;
    QNEP_CUDA_OK(h, cudaMalloc(&h->d_kvec, sizeof(float4) * h->nk));
    QNEP_CUDA_OK(h, cudaMalloc(&h->d_kint, sizeof(int) * h->nk));
    QNEP_CUDA_OK(h, cudaMalloc(&h->d_S, sizeof(double2) * h->nk));
    QNEP_CUDA_OK(h, cudaMalloc(&h->d_ephase, sizeof(float2) * 3 * (size_t)(nm + 1) * h->N));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_kvec, kv.data(), sizeof(float4) * h->nk, cudaMemcpyHostToDevice));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_kint, ki.data(), sizeof(int) * h->nk, cudaMemcpyHostToDevice));
    return QNEP_OK;
}

int qnep_launch_ewald(qnep_handle* h, const double* pos, bool atomv, cudaStream_t s)
{
    const int64_t N = h->N;
    const int addw = h->model.mode == 1 ? 1 : 0;       // mode 1: k_realspace has written the rows of d_Wat
    if (h->nk == 0) {
        if (atomv && !addw) QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_Wat, 0, sizeof(float) * 9 * N, s));
        QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_phik, 0, sizeof(float) * N, s));
        if (h->model.mode != 1) QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_Fs, 0, sizeof(float) * 3 * N, s));
        return QNEP_OK;
    }
    const int nb = (int)((N + 127) / 128);
    k_ewald_phases<<<nb, 128, 0, s>>>(N, pos, h->d_sidx, h->geo, h->ew_nmax, h->d_ephase);
    k_ewald_sfac<<<h->nk, 256, 0, s>>>(N, h->ew_nmax, h->d_ephase, h->d_kint, h->d_q, h->d_S);
    k_ewald_energy<<<std::min(64, (h->nk + 255) / 256), 256, 0, s>>>(h->nk, h->d_kvec, h->d_S, 1.0 / (4.0 * h->alpha * h->alpha),
                                                                    h->d_sums);
    const float inv4a2 = (float)(1.0 / (4.0 * h->alpha * h->alpha));
    if (atomv)
        k_ewald_atoms<true><<<nb, 128, 0, s>>>(N, h->nk, h->ew_nmax, h->d_ephase, h->d_kint, h->d_kvec, h->d_S, h->d_q,
                                               h->model.mode == 1 ? 1 : 0, h->d_phik, h->d_Fs, inv4a2, addw, h->d_Wat);
    else
        k_ewald_atoms<false><<<nb, 128, 0, s>>>(N, h->nk, h->ew_nmax, h->d_ephase, h->d_kint, h->d_kvec, h->d_S, h->d_q,
                                                h->model.mode == 1 ? 1 : 0, h->d_phik, h->d_Fs, inv4a2, 0, nullptr);
    h->launches += 4;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}
