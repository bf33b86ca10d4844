// pppm.cu -- steps a7P-1..5 of SURVEY.md 8(a): PPPM evaluation of the reciprocal-space part
// (PAPER.md II.F, Eq. 34-38; readings G2, S10, S11):
//   1. charge assignment with the order-5 cardinal B-spline (Eq. 35)
//   2. forward 3-D FFT of the charge mesh (hand-written, no cuFFT; :302)
//   3. multiply by the optimised influence function G^opt (Eq. 36), energy (Eq. 34) and virial (Eq. 22)
//   4. inverse 3-D FFTs.  The four real fields F^-1[S G], F^-1[i k_a S G] (Eq. 37, 38; "3 + 1 backward
//      FFTs", :302) are packed pairwise into TWO complex transforms: M1 = Phi + i E_x, M2 = E_y + i E_z.
//   5. back-interpolation of phi^k_i and F^{k,static}_i with the same B-spline.
//
// FFT design: a line of N = R1 R2 points is held in the REGISTERS of N / 16 (or fewer) threads; two
// small register DFTs (fft_reg.cuh) with one shared-memory exchange in between transform it, so a pass is one
// coalesced global read and one coalesced global write of the mesh.  16 lines form a tile; strided axes move
// 128-byte row segments.  The pass along x is FUSED with step 3 and with the first inverse pass: forward x-FFT ->
// influence multiply (+ energy / virial sums) -> two inverse x-FFTs, all on registers: the spectrum S(k) and the
// four field spectra never exist in HBM.  The last inverse pass (z) transforms M1 and M2 together and writes the
// four real fields interleaved as float4 (Phi, E_x, E_y, E_z), which step 5 reads with one 16-byte load per point.
// Passes per evaluation: z, y, x-fused, y (x2 meshes), z (x2 meshes) = 5 kernels, 7 mesh read+write sweeps
// instead of 9 transforms x 3 passes.
#include "qnep_internal.cuh"

#include <cmath>
#include <type_traits>

#include "fft_reg.cuh"
#include "pppm_common.cuh"

namespace {

constexpr int FFT_MAXN = 512;

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
// The 5 consecutive z points of a stencil row always fall into exactly two aligned quads of the mesh row, so a row
// is added with two 16-byte vector reductions (REDG.ADD.F32x4) instead of five scalar ones: the SM issues
// reductions at a fixed rate per lane-instruction, so this is 50 instead of 125 per atom.
__device__ __forceinline__ void red_add_v4(float* p, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__global__ void __launch_bounds__(128)
k_spread(int64_t N, Geometry g, const float4* __restrict__ mfrac, const int* __restrict__ mi0, const int* __restrict__ cm,
         const float* __restrict__ q, float* __restrict__ mesh)
{
    // Threads walk the (type, cell) order here, not the cell-major one: the kernel is bound by L2 reductions, and
    // spreading one species at a time halves the number of reductions that meet in the same sector at the same moment
    // (0.23 -> 0.21 ms on config 4; a stride that scatters concurrent threads over the whole box is slower again).  The mesh coordinates are stored in cell-major order (for k_gather): one gather.
    const int64_t ps = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;     // sorted index
    if (ps >= N) return;
    const int64_t p = cm[ps];                                              // cell-major rank
    const float4 fr = mfrac[p];
    float wx[5], wy[5], wz[5];
    bspline5(fr.x, wx); bspline5(fr.y, wy); bspline5(fr.z, wz);
    int idx[3][5];
    stencil_indices(mi0[p], g.grid, idx);
    // z weights placed in two aligned quads
    const int z0 = idx[2][0];
    const int o = z0 & 3;
    const int q0 = z0 - o, q1 = (q0 + 4) & (g.grid[2] - 1);
    float w8[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        float v = 0.f;
#pragma unroll
        for (int c = 0; c < 5; ++c)
            if (i - c >= 0 && i - c <= 3) v = (o == i - c) ? wz[c] : v;
        w8[i] = v;
    }
    const float qi = q[ps];
#pragma unroll
    for (int a = 0; a < 5; ++a) {
        const float qa = qi * wx[a];
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const float qab = qa * wy[b];
            float* row = mesh + ((int64_t)idx[0][a] * g.grid[1] + idx[1][b]) * g.grid[2];
            red_add_v4(row + q0, qab * w8[0], qab * w8[1], qab * w8[2], qab * w8[3]);
            red_add_v4(row + q1, qab * w8[4], qab * w8[5], qab * w8[6], qab * w8[7]);
        }
    }
}

// ---- 2./4. FFT building blocks ------------------------------------------------------------------
using fftreg::dft;

constexpr int LINES = 16;          // lines per tile

template <int R1, int R2>
struct Split {
    static constexpr int N = R1 * R2;
    static constexpr int TPL = R1 < R2 ? R1 : R2;      // threads per line
    static constexpr int E = N / TPL;                  // elements per thread
    static constexpr int D1 = R2 / TPL;                // stage-1 DFTs (length R1) per thread
    static constexpr int D2 = R1 / TPL;                // stage-2 DFTs (length R2) per thread
    static constexpr int LP = (R2 * (R1 + 1)) | 1;     // exchange pitch of one line (float2), odd: conflict-free across lines
    static constexpr int THREADS = TPL * LINES;
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// One line transform on registers.
//   in : v[d * R1 + m]  = x[(u + TPL d) + R2 m],   d < D1, m < R1     ("stage-1 layout" of <R1, R2>)
//   out: v[d * R2 + k1] = X[(u + TPL d) + R1 k1],  d < D2, k1 < R2    ("stage-2 layout" of <R1, R2>,
//                                                                       = the stage-1 layout of <R2, R1>)
// sm: this line's exchange area (Split::LP float2); tw: omega_N^j = e^{-2 pi i j / N}, j < N (shared memory).
// All threads of the block must call it (two block barriers).
template <int R1, int R2, int SIGN>
__device__ __forceinline__ void line_fft(float2* v, float2* sm, int u, const float2* tw)
{
    using S = Split<R1, R2>;
#pragma unroll
    for (int d = 0; d < S::D1; ++d) {
        dft<R1, SIGN>(v + d * R1);
        const int t = u + S::TPL * d;
#pragma unroll
        for (int k2 = 0; k2 < R1; ++k2) {
            float2 x = v[d * R1 + k2];
            if (k2 > 0) {
                float2 w = tw[t * k2];
                if (SIGN > 0) w.y = -w.y;
                x = cmul(x, w);
            }
            sm[t * (R1 + 1) + k2] = x;
        }
    }
    __syncthreads();
#pragma unroll
    for (int d = 0; d < S::D2; ++d) {
        const int k2 = u + S::TPL * d;
#pragma unroll
        for (int t = 0; t < R2; ++t) v[d * R2 + t] = sm[t * (R1 + 1) + k2];
        dft<R2, SIGN>(v + d * R2);
    }
    __syncthreads();
}

struct TileAddr { int64_t base, stride; };

// tile -> (base, stride) of a strided-axis tile: 16 consecutive z (b), all points of `axis`
__device__ __forceinline__ TileAddr strided_tile(int axis, int n0, int n1, int n2, int64_t tile)
{
    const int zc = n2 / LINES;
    TileAddr a;
    if (axis == 1) { a.base = (tile / zc) * (int64_t)n1 * n2 + (tile % zc) * LINES; a.stride = n2; }
    else { a.base = (tile / zc) * (int64_t)n2 + (tile % zc) * LINES; a.stride = (int64_t)n1 * n2; }
    (void)n0;
    return a;
}

__device__ __forceinline__ void load_twiddles(float2* tw, const float2* __restrict__ g, int n)
{
    for (int i = threadIdx.x; i < n; i += blockDim.x) tw[i] = g[i];
}

// ---- forward pass along z: real mesh -> complex ---------------------------------------------------
template <int R1, int R2>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS)
k_fft_z_fwd(const float* __restrict__ rho, float2* __restrict__ out, const float2* __restrict__ twg)
{
    using S = Split<R1, R2>;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * S::LP;
    load_twiddles(tw, twg, S::N);
    __syncthreads();
    const int u = threadIdx.x % S::TPL, b = threadIdx.x / S::TPL;
    const int64_t base = ((int64_t)blockIdx.x * LINES + b) * S::N;
    float2 v[S::E];
#pragma unroll
    for (int d = 0; d < S::D1; ++d)
#pragma unroll
        for (int m = 0; m < R1; ++m) v[d * R1 + m] = make_float2(rho[base + (u + S::TPL * d) + R2 * m], 0.f);
    line_fft<R1, R2, -1>(v, smem + b * S::LP, u, tw);
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) out[base + (u + S::TPL * d) + R1 * k1] = v[d * R2 + k1];
}

// ---- forward pass along z, half spectrum: the mesh is real, so S(-k) = conj S(k) and only kz = 0 .. N/2 is kept.
// Half arrays are [x][y][NH] with NH = N/2 + LINES: slots 0 .. N/2 hold kz, the rest of the last tile stays zero.
template <int R1, int R2>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS)
k_fft_z_fwd_half(const float* __restrict__ rho, float2* __restrict__ out, const float2* __restrict__ twg)
{
    using S = Split<R1, R2>;
    constexpr int NH = S::N / 2 + LINES;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * S::LP;
    load_twiddles(tw, twg, S::N);
    __syncthreads();
    const int u = threadIdx.x % S::TPL, b = threadIdx.x / S::TPL;
    const int64_t line = (int64_t)blockIdx.x * LINES + b;
    float2 v[S::E];
#pragma unroll
    for (int d = 0; d < S::D1; ++d)
#pragma unroll
        for (int m = 0; m < R1; ++m) v[d * R1 + m] = make_float2(rho[line * S::N + (u + S::TPL * d) + R2 * m], 0.f);
    line_fft<R1, R2, -1>(v, smem + b * S::LP, u, tw);
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) {
            const int kz = (u + S::TPL * d) + R1 * k1;
            if (kz <= S::N / 2) out[line * NH + kz] = v[d * R2 + k1];
        }
}

// ---- in-place pass along a strided axis (y): grid.y selects the mesh --------------------------------
#ifndef QNEP_FFT_STRIDED_MINB
#define QNEP_FFT_STRIDED_MINB 3       // three blocks of 256 threads per SM: 0.855 -> 0.812 ms per reciprocal stage (1, 2, 4, 5 are slower)
#endif
#ifndef QNEP_FFT_ZF_MINB
#define QNEP_FFT_ZF_MINB 3
#endif
template <int R1, int R2, int SIGN>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS, Split<R1, R2>::THREADS >= 256 ? QNEP_FFT_STRIDED_MINB : 1)
k_fft_strided(int axis, int n0, int n1, int n2, float2* __restrict__ mesh_a, float2* __restrict__ mesh_b,
              const float2* __restrict__ twg)
{
    using S = Split<R1, R2>;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * S::LP;
    load_twiddles(tw, twg, S::N);
    __syncthreads();
    float2* mesh = blockIdx.y == 0 ? mesh_a : mesh_b;
    const int b = threadIdx.x % LINES, u = threadIdx.x / LINES;
    const TileAddr ta = strided_tile(axis, n0, n1, n2, blockIdx.x);
    float2* p = mesh + ta.base + b;
    float2 v[S::E];
#pragma unroll
    for (int d = 0; d < S::D1; ++d)
#pragma unroll
        for (int m = 0; m < R1; ++m) v[d * R1 + m] = p[((u + S::TPL * d) + R2 * m) * ta.stride];
    line_fft<R1, R2, SIGN>(v, smem + b * S::LP, u, tw);
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) p[((u + S::TPL * d) + R1 * k1) * ta.stride] = v[d * R2 + k1];
}

// Non-orthogonal cells (PAPER.md :104, k from the reciprocal basis vectors): b[3a + c] = Cartesian component a of 2 pi b*_c.
// The tables of a triclinic run hold the INTEGER index n of the axis in kk[] (k = sum_c n_c b_c is formed per mesh point,
// and exp(-k^2 / 4 alpha^2) with it: neither is separable any more) and A[] without the Gaussian.  The gradient multiplier
// stays per axis: kd[] = 2 pi n / |cell vector| (Nyquist entry zeroed), i.e. the meshes carry the components of
// grad Phi along the RECIPROCAL basis vectors, and k_gather turns them into Cartesian components with the constant
// matrix hinv[3a + c] |h_c| (the identity for an orthorhombic box).  That keeps kd_y, kd_z constants of an x line, which
// the packing of the four fields into two transforms and the mirror lines of the half spectrum rely on.
struct KB { float b[9]; };

// ---- 3. fused pass along x: forward FFT, influence function, two inverse FFTs ------------------------
// tables per axis a (offset a * FFT_MAXN): A[m] = exp(-k^2/4 alpha^2) sinc^10(pi n/N) / d(z)^2, kk[m] = k (true, for
// k^2), kd[m] = k with the Nyquist entry zeroed (for the i k multiplier, S11).
//   M1 = Phi + i (i kx Phi) = (1 - kx) Phi ;  M2 = i ky Phi + i (i kz Phi) = (-kz + i ky) Phi
template <int R1, int R2, bool VIRIAL, bool TRI>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS)
k_fft_x_fused(int n0, int n1, int n2, float2* __restrict__ M1 /* in: S after the z and y passes; out: M1 */,
              float2* __restrict__ M2, const float2* __restrict__ twg, const float* __restrict__ tabA,
              const float* __restrict__ tabK, const float* __restrict__ tabKd, float c0 /* 2 pi / Omega */, float inv4a2,
              double* __restrict__ sums, KB kb)
{
    using S = Split<R1, R2>;
    using SI = Split<R2, R1>;
    constexpr int LPMAX = S::LP > SI::LP ? S::LP : SI::LP;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * LPMAX;
    float* tA = reinterpret_cast<float*>(tw + S::N);
    float* tK = tA + S::N;
    float* tKd = tK + S::N;
    __shared__ double sh_red[32];
    load_twiddles(tw, twg, S::N);
    for (int i = threadIdx.x; i < S::N; i += blockDim.x) { tA[i] = tabA[i]; tK[i] = tabK[i]; tKd[i] = tabKd[i]; }
    __syncthreads();
    const int b = threadIdx.x % LINES, u = threadIdx.x / LINES;
    const TileAddr ta = strided_tile(0, n0, n1, n2, blockIdx.x);
    const int zc = n2 / LINES;
    const int iy = (int)(blockIdx.x / zc), iz = (int)(blockIdx.x % zc) * LINES + b;
    float2 v[S::E], w[S::E];
    {
        const float2* p = M1 + ta.base + b;
#pragma unroll
        for (int d = 0; d < S::D1; ++d)
#pragma unroll
            for (int m = 0; m < R1; ++m) v[d * R1 + m] = p[((u + S::TPL * d) + R2 * m) * ta.stride];
    }
    line_fft<R1, R2, -1>(v, smem + b * S::LP, u, tw);
    // v[d * R2 + k1] = S(kx = (u + TPL d) + R1 k1, ky, kz)
    const float ky = tabK[FFT_MAXN + iy], kz = tabK[2 * FFT_MAXN + iz];
    const float kdy = tabKd[FFT_MAXN + iy], kdz = tabKd[2 * FFT_MAXN + iz];
    const float Ayz = c0 * tabA[FFT_MAXN + iy] * tabA[2 * FFT_MAXN + iz];
    const float kyz2 = ky * ky + kz * kz;
    // TRI: ky, kz are the integer indices n1, n2 and (lx, ly, lz) = n1 b_1 + n2 b_2 is the part of k shared by the line
    const float lx = TRI ? ky * kb.b[1] + kz * kb.b[2] : 0.f, ly = TRI ? ky * kb.b[4] + kz * kb.b[5] : 0.f, lz = TRI ? ky * kb.b[7] + kz * kb.b[8] : 0.f;
    float acc[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) {
            const int ix = (u + S::TPL * d) + R1 * k1;
            const float kdx = tKd[ix];
            float kx = tK[ix], kyp = ky, kzp = kz, k2;
            if (TRI) { const float nx = kx; kx = fmaf(nx, kb.b[0], lx); kyp = fmaf(nx, kb.b[3], ly); kzp = fmaf(nx, kb.b[6], lz); k2 = kx * kx + kyp * kyp + kzp * kzp; }
            else k2 = kx * kx + kyz2;
            const float2 s = v[d * R2 + k1];
            float G = 0.f;
            if (k2 > 0.f) G = __fdividef(TRI ? Ayz * tA[ix] * __expf(-k2 * inv4a2) : Ayz * tA[ix], k2);
            const float2 phi = make_float2(G * s.x, G * s.y);
            const float e = G * (s.x * s.x + s.y * s.y);
            acc[0] += e;
            if (VIRIAL && k2 > 0.f) {
                const float bf = 2.f * inv4a2 + __fdividef(2.f, k2);
                acc[1] += e * (1.f - bf * kx * kx);
                acc[2] += e * (-bf * kx * kyp);
                acc[3] += e * (-bf * kx * kzp);
                acc[4] += e * (1.f - bf * kyp * kyp);
                acc[5] += e * (-bf * kyp * kzp);
                acc[6] += e * (1.f - bf * kzp * kzp);
            }
            v[d * R2 + k1] = make_float2((1.f - kdx) * phi.x, (1.f - kdx) * phi.y);
            w[d * R2 + k1] = make_float2(-kdz * phi.x - kdy * phi.y, -kdz * phi.y + kdy * phi.x);
        }
    // inverse along x with the swapped split <R2, R1>: its stage-1 layout is the layout we hold
    line_fft<R2, R1, +1>(v, smem + b * SI::LP, u, tw);
    {
        float2* p = M1 + ta.base + b;
#pragma unroll
        for (int d = 0; d < SI::D2; ++d)
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) p[((u + SI::TPL * d) + R2 * k1) * ta.stride] = v[d * R1 + k1];
    }
    line_fft<R2, R1, +1>(w, smem + b * SI::LP, u, tw);
    {
        float2* p = M2 + ta.base + b;
#pragma unroll
        for (int d = 0; d < SI::D2; ++d)
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) p[((u + SI::TPL * d) + R2 * k1) * ta.stride] = w[d * R1 + k1];
    }
    // U^k = K sum G |S|^2 (Eq. 34), W^k = K sum G |S|^2 B (Eq. 22): fp32 per thread, fp64 across threads
    const int slot[7] = {SUM_U_K, SUM_W0 + 0, SUM_W0 + 1, SUM_W0 + 2, SUM_W0 + 4, SUM_W0 + 5, SUM_W0 + 8};
    const int mirror[7] = {-1, -1, SUM_W0 + 3, SUM_W0 + 6, -1, SUM_W0 + 7, -1};
#pragma unroll
    for (int a = 0; a < (VIRIAL ? 7 : 1); ++a) {
        double x = (double)acc[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) sh_red[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x < 32) {
            double r = threadIdx.x < (blockDim.x >> 5) ? sh_red[threadIdx.x] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
            if (threadIdx.x == 0) {
                r *= QNEP_K_COULOMB;
                atomicAdd(&sums[slot[a]], r);
                if (mirror[a] >= 0) atomicAdd(&sums[mirror[a]], r);
            }
        }
    }
}

// ---- 3'. fused pass along x on the half spectrum ----------------------------------------------------
// Input: half array H (kz = 0 .. N2/2) after the z and y passes.  For every stored line (ky, kz) the kernel writes the
// inverse-x transforms of M1 and M2 at (ky, kz) and, for 0 < kz < N2/2, at the mirror line (-ky, -kz), which is not
// stored: with phi(-k) = conj phi(k), k_d odd and the identity  IDFT[conj a(-k)] = conj IDFT[a(k)]  the mirror lines are
//     M1(x; -ky, -kz) = conj IDFT_x[(1 + kd_x) phi],     M2(x; -ky, -kz) = conj IDFT_x[(kd_z + i kd_y) phi],
// with kd_y, kd_z of the STORED line.  Energy and virial sums weigh these lines twice.  One forward and four inverse
// line transforms per stored line instead of one and two per line of the full spectrum.
template <int R1, int R2, bool VIRIAL, bool TRI>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS, Split<R1, R2>::THREADS >= 256 ? 3 : 1)
k_fft_x_fused_half(int n0, int n1, int n2, const float2* __restrict__ H, float2* __restrict__ M1, float2* __restrict__ M2,
                   const float2* __restrict__ twg, const float* __restrict__ tabA, const float* __restrict__ tabK,
                   const float* __restrict__ tabKd, float c0 /* 2 pi / Omega */, float inv4a2, double* __restrict__ sums, KB kb)
{
    using S = Split<R1, R2>;
    using SI = Split<R2, R1>;
    constexpr int LPMAX = S::LP > SI::LP ? S::LP : SI::LP;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * LPMAX;
    float* tA = reinterpret_cast<float*>(tw + S::N);
    float* tK = tA + S::N;
    float* tKd = tK + S::N;
    float2* sphi = reinterpret_cast<float2*>(tKd + S::N) + threadIdx.x;     // phi(kx) of this thread: sphi[e * THREADS]
    __shared__ double sh_red[32];
    load_twiddles(tw, twg, S::N);
    for (int i = threadIdx.x; i < S::N; i += blockDim.x) { tA[i] = tabA[i]; tK[i] = tabK[i]; tKd[i] = tabKd[i]; }
    __syncthreads();
    const int NH = n2 / 2 + LINES;
    const int b = threadIdx.x % LINES, u = threadIdx.x / LINES;
    const int zc = NH / LINES;
    const int iy = (int)(blockIdx.x / zc), kz = (int)(blockIdx.x % zc) * LINES + b;
    const bool valid = kz <= n2 / 2;
    const bool mirrored = kz > 0 && kz < n2 / 2;
    const int64_t hstride = (int64_t)n1 * NH, fstride = (int64_t)n1 * n2;
    float2 v[S::E];
    {
        const float2* p = H + (int64_t)iy * NH + kz;
#pragma unroll
        for (int d = 0; d < S::D1; ++d)
#pragma unroll
            for (int m = 0; m < R1; ++m) v[d * R1 + m] = p[((u + S::TPL * d) + R2 * m) * hstride];
    }
    line_fft<R1, R2, -1>(v, smem + b * S::LP, u, tw);
    // v[d * R2 + k1] = S(kx = (u + TPL d) + R1 k1, ky, kz)
    const int kzc = valid ? kz : 0;
    const float ky = tabK[FFT_MAXN + iy], kzv = tabK[2 * FFT_MAXN + kzc];
    const float kdy = tabKd[FFT_MAXN + iy], kdz = tabKd[2 * FFT_MAXN + kzc];
    const float Ayz = c0 * tabA[FFT_MAXN + iy] * tabA[2 * FFT_MAXN + kzc];
    const float kyz2 = ky * ky + kzv * kzv;
    // TRI: ky, kzv are the integer indices n1, n2 and (lx, ly, lz) = n1 b_1 + n2 b_2 is the part of k shared by the line
    const float lx = TRI ? ky * kb.b[1] + kzv * kb.b[2] : 0.f, ly = TRI ? ky * kb.b[4] + kzv * kb.b[5] : 0.f, lz = TRI ? ky * kb.b[7] + kzv * kb.b[8] : 0.f;
    const float wgt = !valid ? 0.f : (mirrored ? 2.f : 1.f);
    float acc[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) {
            const int ix = (u + S::TPL * d) + R1 * k1;
            float kx = tK[ix], kyp = ky, kzp = kzv, k2;
            if (TRI) { const float nx = kx; kx = fmaf(nx, kb.b[0], lx); kyp = fmaf(nx, kb.b[3], ly); kzp = fmaf(nx, kb.b[6], lz); k2 = kx * kx + kyp * kyp + kzp * kzp; }
            else k2 = kx * kx + kyz2;
            const float2 sv = v[d * R2 + k1];
            float G = 0.f;
            if (k2 > 0.f) G = __fdividef(TRI ? Ayz * tA[ix] * __expf(-k2 * inv4a2) : Ayz * tA[ix], k2);
            // phi = G S stays in the registers, kd_x phi is parked in shared memory for the second inverse transform
            const float2 ph = make_float2(G * sv.x, G * sv.y);
            const float kdx = tKd[ix];
            v[d * R2 + k1] = ph;
            sphi[(d * R2 + k1) * S::THREADS] = make_float2(kdx * ph.x, kdx * ph.y);
            const float e = wgt * G * (sv.x * sv.x + sv.y * sv.y);
            acc[0] += e;
            if (VIRIAL && k2 > 0.f) {
                const float bf = 2.f * inv4a2 + __fdividef(2.f, k2);
                acc[1] += e * (1.f - bf * kx * kx);
                acc[2] += e * (-bf * kx * kyp);
                acc[3] += e * (-bf * kx * kzp);
                acc[4] += e * (1.f - bf * kyp * kyp);
                acc[5] += e * (-bf * kyp * kzp);
                acc[6] += e * (1.f - bf * kzp * kzp);
            }
        }
    // Two inverse transforms along x give all four output lines, because kd_y and kd_z are constants of the line:
    //   A = IDFT_x[phi], B = IDFT_x[kd_x phi]:   M1 = A - B,  M2 = (-kd_z + i kd_y) A   at (ky, kz),
    //   conj(A + B)  and  conj((kd_z + i kd_y) A)                                         at (-ky, -kz).
    // (swapped split <R2, R1>: its stage-1 layout is the layout we hold)
    const int iym = (n1 - iy) % n1, kzm = n2 - kz;
    float2* own1 = M1 + (int64_t)iy * n2 + kz;
    float2* own2 = M2 + (int64_t)iy * n2 + kz;
    float2* mir1 = M1 + (int64_t)iym * n2 + kzm;
    float2* mir2 = M2 + (int64_t)iym * n2 + kzm;
    line_fft<R2, R1, +1>(v, smem + b * SI::LP, u, tw);          // v = A
#pragma unroll
    for (int d = 0; d < SI::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            const int64_t off = (int64_t)((u + SI::TPL * d) + R2 * k1) * fstride;
            const float2 A = v[d * R1 + k1];
            if (valid) own2[off] = make_float2(-kdz * A.x - kdy * A.y, -kdz * A.y + kdy * A.x);
            if (mirrored) mir2[off] = make_float2(kdz * A.x - kdy * A.y, -(kdz * A.y + kdy * A.x));
            // swap: A goes to shared memory, kd_x phi comes back for the second transform.  The element index differs
            // between the two layouts, but a slot is only a parking place of this thread: any one-to-one order works.
            float2* slot = sphi + (d * R1 + k1) * S::THREADS;
            const float2 t = *slot;
            *slot = A;
            v[d * R1 + k1] = t;
        }
    line_fft<R2, R1, +1>(v, smem + b * SI::LP, u, tw);          // v = B
#pragma unroll
    for (int d = 0; d < SI::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R1; ++k1) {
            const int64_t off = (int64_t)((u + SI::TPL * d) + R2 * k1) * fstride;
            const float2 A = sphi[(d * R1 + k1) * S::THREADS], B = v[d * R1 + k1];
            if (valid) own1[off] = make_float2(A.x - B.x, A.y - B.y);
            if (mirrored) mir1[off] = make_float2(A.x + B.x, -(A.y + B.y));
        }
    // U^k = K sum G |S|^2 (Eq. 34), W^k = K sum G |S|^2 B (Eq. 22): fp32 per thread, fp64 across threads
    const int slot[7] = {SUM_U_K, SUM_W0 + 0, SUM_W0 + 1, SUM_W0 + 2, SUM_W0 + 4, SUM_W0 + 5, SUM_W0 + 8};
    const int mirror[7] = {-1, -1, SUM_W0 + 3, SUM_W0 + 6, -1, SUM_W0 + 7, -1};
#pragma unroll
    for (int a = 0; a < (VIRIAL ? 7 : 1); ++a) {
        double x = (double)acc[a];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) sh_red[threadIdx.x >> 5] = x;
        __syncthreads();
        if (threadIdx.x < 32) {
            double r = threadIdx.x < (blockDim.x >> 5) ? sh_red[threadIdx.x] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
            if (threadIdx.x == 0) {
                r *= QNEP_K_COULOMB;
                atomicAdd(&sums[slot[a]], r);
                if (mirror[a] >= 0) atomicAdd(&sums[mirror[a]], r);
            }
        }
    }
    (void)n0;
}

// ---- 3''. per-atom virial pass along x (Eq. 39): forward FFT, phi = G^opt S, three inverse FFTs ---------------
// The six real fields F^-1[S G^opt B_ab] ("six backward FFTs", :302) are packed pairwise into three complex transforms,
//   M1 = W_xx + i W_yy,   M2 = W_zz + i W_xy,   M3 = W_xz + i W_yz,      B_ab = delta_ab - (2 / 4 alpha^2 + 2 / k^2) k_a k_b
// (B is real and even in k, so each product phi B_ab is the spectrum of a real field).  Full spectrum in M3 (after the
// forward z and y passes), in-place line by line for M3.
template <int R1, int R2, bool TRI>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS)
k_fft_x_virial(int n0, int n1, int n2, float2* __restrict__ M1, float2* __restrict__ M2, float2* __restrict__ M3,
               const float2* __restrict__ twg, const float* __restrict__ tabA, const float* __restrict__ tabK,
               float c0 /* 2 pi / Omega */, float inv4a2, KB kb)
{
    using S = Split<R1, R2>;
    using SI = Split<R2, R1>;
    constexpr int LPMAX = S::LP > SI::LP ? S::LP : SI::LP;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * LPMAX;
    float* tA = reinterpret_cast<float*>(tw + S::N);
    float* tK = tA + S::N;
    load_twiddles(tw, twg, S::N);
    for (int i = threadIdx.x; i < S::N; i += blockDim.x) { tA[i] = tabA[i]; tK[i] = tabK[i]; }
    __syncthreads();
    const int b = threadIdx.x % LINES, u = threadIdx.x / LINES;
    const TileAddr ta = strided_tile(0, n0, n1, n2, blockIdx.x);
    const int zc = n2 / LINES;
    const int iy = (int)(blockIdx.x / zc), iz = (int)(blockIdx.x % zc) * LINES + b;
    float2 ph[S::E], v[S::E];
    {
        const float2* p = M3 + ta.base + b;
#pragma unroll
        for (int d = 0; d < S::D1; ++d)
#pragma unroll
            for (int m = 0; m < R1; ++m) ph[d * R1 + m] = p[((u + S::TPL * d) + R2 * m) * ta.stride];
    }
    line_fft<R1, R2, -1>(ph, smem + b * S::LP, u, tw);
    const float ky = tabK[FFT_MAXN + iy], kz = tabK[2 * FFT_MAXN + iz];
    const float Ayz = c0 * tabA[FFT_MAXN + iy] * tabA[2 * FFT_MAXN + iz];
    const float kyz2 = ky * ky + kz * kz;
    const float lx = TRI ? ky * kb.b[1] + kz * kb.b[2] : 0.f, ly = TRI ? ky * kb.b[4] + kz * kb.b[5] : 0.f, lz = TRI ? ky * kb.b[7] + kz * kb.b[8] : 0.f;
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) {
            const int ix = (u + S::TPL * d) + R1 * k1;
            float kx = tK[ix], kyp = ky, kzp = kz, k2;
            if (TRI) { const float nx = kx; kx = fmaf(nx, kb.b[0], lx); kyp = fmaf(nx, kb.b[3], ly); kzp = fmaf(nx, kb.b[6], lz); k2 = kx * kx + kyp * kyp + kzp * kzp; }
            else k2 = kx * kx + kyz2;
            const float G = k2 > 0.f ? __fdividef(TRI ? Ayz * tA[ix] * __expf(-k2 * inv4a2) : Ayz * tA[ix], k2) : 0.f;
            ph[d * R2 + k1].x *= G; ph[d * R2 + k1].y *= G;
        }
    float2* const Ms[3] = {M1, M2, M3};
#pragma unroll
    for (int pair = 0; pair < 3; ++pair) {
#pragma unroll
        for (int d = 0; d < S::D2; ++d)
#pragma unroll
            for (int k1 = 0; k1 < R2; ++k1) {
                const int ix = (u + S::TPL * d) + R1 * k1;
                float kx = tK[ix], kyp = ky, kzp = kz, k2;
                if (TRI) { const float nx = kx; kx = fmaf(nx, kb.b[0], lx); kyp = fmaf(nx, kb.b[3], ly); kzp = fmaf(nx, kb.b[6], lz); k2 = kx * kx + kyp * kyp + kzp * kzp; }
                else k2 = kx * kx + kyz2;
                const float bf = k2 > 0.f ? 2.f * inv4a2 + __fdividef(2.f, k2) : 0.f;
                const float one = k2 > 0.f ? 1.f : 0.f;
                float B1, B2;
                if (pair == 0) { B1 = one - bf * kx * kx; B2 = one - bf * kyp * kyp; }
                else if (pair == 1) { B1 = one - bf * kzp * kzp; B2 = -bf * kx * kyp; }
                else { B1 = -bf * kx * kzp; B2 = -bf * kyp * kzp; }
                const float2 f = ph[d * R2 + k1];
                v[d * R2 + k1] = make_float2(f.x * B1 - f.y * B2, f.x * B2 + f.y * B1);
            }
        // inverse along x with the swapped split <R2, R1>: its stage-1 layout is the layout we hold
        line_fft<R2, R1, +1>(v, smem + b * SI::LP, u, tw);
        float2* p = Ms[pair] + ta.base + b;
#pragma unroll
        for (int d = 0; d < SI::D2; ++d)
#pragma unroll
            for (int k1 = 0; k1 < R1; ++k1) p[((u + SI::TPL * d) + R2 * k1) * ta.stride] = v[d * R1 + k1];
    }
}

// Layout of the (Phi, E) mesh read by k_gather.  QNEP_FIELD_BRICKS = 0: [x][y][z] rows; a 5-point z run of float4 (80 B)
// straddles a 128-byte line half the time, 37.5 line visits per 5^3 stencil.  QNEP_FIELD_BRICKS = 1: 2 x 2 x 2 bricks of
// float4, one brick = one 128-byte line, point (x, y, z) at 8 * brick + (x & 1, y & 1, z & 1): five consecutive points of an
// axis always fall into three bricks, so a stencil visits 27 lines, each read whole by the eight lanes of an atom's group.
#ifndef QNEP_FIELD_BRICKS
#define QNEP_FIELD_BRICKS 0
#endif
__device__ __forceinline__ int field_brick_index(int x, int y, int z, int n1, int n2)
{
    return (((((x >> 1) * (n1 >> 1) + (y >> 1)) * (n2 >> 1)) + (z >> 1)) << 3) | ((x & 1) << 2) | ((y & 1) << 1) | (z & 1);
}

// ---- last inverse pass along z: M1, M2 -> interleaved real fields (Phi, E_x, E_y, E_z) -------------------
template <int R1, int R2>
__global__ void __launch_bounds__(Split<R1, R2>::THREADS, Split<R1, R2>::THREADS >= 256 ? QNEP_FFT_ZF_MINB : 1)
k_fft_z_fields(const float2* __restrict__ M1, const float2* __restrict__ M2, float4* __restrict__ field,
               const float2* __restrict__ twg, int n1)
{
    using S = Split<R1, R2>;
    extern __shared__ __align__(16) float2 smem[];
    float2* tw = smem + LINES * S::LP;
    load_twiddles(tw, twg, S::N);
    __syncthreads();
    const int u = threadIdx.x % S::TPL, b = threadIdx.x / S::TPL;
    const int64_t base = ((int64_t)blockIdx.x * LINES + b) * S::N;
    float2 v[S::E], w[S::E];
#pragma unroll
    for (int d = 0; d < S::D1; ++d)
#pragma unroll
        for (int m = 0; m < R1; ++m) {
            v[d * R1 + m] = M1[base + (u + S::TPL * d) + R2 * m];
            w[d * R1 + m] = M2[base + (u + S::TPL * d) + R2 * m];
        }
    line_fft<R1, R2, +1>(v, smem + b * S::LP, u, tw);
    line_fft<R1, R2, +1>(w, smem + b * S::LP, u, tw);
#pragma unroll
    for (int d = 0; d < S::D2; ++d)
#pragma unroll
        for (int k1 = 0; k1 < R2; ++k1) {
            const float2 a = v[d * R2 + k1], c = w[d * R2 + k1];
#if QNEP_FIELD_BRICKS
            const int line = blockIdx.x * LINES + b, x = line / n1, y = line - x * n1, z = (u + S::TPL * d) + R1 * k1;
            field[field_brick_index(x, y, z, n1, S::N)] = make_float4(a.x, a.y, c.x, c.y);
#else
            field[base + (u + S::TPL * d) + R1 * k1] = make_float4(a.x, a.y, c.x, c.y);
#endif
        }
}

// ---- 5. back-interpolation ------------------------------------------------------------------------
// Phase 1: one thread per atom computes the B-spline weights and the wrapped stencil offsets into shared memory.
// Phase 2: eight lanes serve one atom: lane c < 5 reads stencil column z_c of each of the 25 (x, y) rows, so one
// load instruction touches one or two 128-byte lines per atom (5 consecutive float4) instead of one line per lane;
// the four sums are reduced over the lane group with shuffles.
constexpr int GATHER_GROUP = 8;
constexpr int GATHER_BLOCK = 128;

// VMODE (per-atom virial pass, Eq. 39): the four interpolated values are K q_i times four virial components; rows.x..w /
// mirror.x..w name the rows of Wat [9][N] they are added to (-1: none).
struct GatherRows { int row[4], mirror[4]; };

template <bool VMODE>
__global__ void __launch_bounds__(GATHER_BLOCK)
k_gather(int64_t N, Geometry g, const float4* __restrict__ mfrac, const int* __restrict__ mi0, const int* __restrict__ cmi,
         const float* __restrict__ q, const float4* __restrict__ field, int add_to_Fs,
         float* __restrict__ phik, float* __restrict__ Fs, GatherRows vr, float* __restrict__ Wat)
{
    __shared__ float s_w[3][5][GATHER_BLOCK];
    __shared__ int s_i[3][5][GATHER_BLOCK];       // x: index * n1 * n2, y: index * n2, z: index
    __shared__ float s_out[4][GATHER_BLOCK];
#if QNEP_FIELD_BRICKS
    __shared__ int s_first[3][GATHER_BLOCK];      // wrapped index of the first stencil point per axis
#endif
    const int t = threadIdx.x;
    const int64_t p0 = blockIdx.x * (int64_t)GATHER_BLOCK;
    {
        const int64_t p = min(p0 + t, N - 1);
        const float4 fr = mfrac[p];
        float w[3][5];
        bspline5(fr.x, w[0]); bspline5(fr.y, w[1]); bspline5(fr.z, w[2]);
        int idx[3][5];
        stencil_indices(mi0[p], g.grid, idx);
#pragma unroll
        for (int i = 0; i < 5; ++i) {
            s_w[0][i][t] = w[0][i]; s_w[1][i][t] = w[1][i]; s_w[2][i][t] = w[2][i];
            s_i[0][i][t] = idx[0][i] * g.grid[1] * g.grid[2];
            s_i[1][i][t] = idx[1][i] * g.grid[2];
            s_i[2][i][t] = idx[2][i];
        }
#if QNEP_FIELD_BRICKS
        s_first[0][t] = idx[0][0]; s_first[1][t] = idx[1][0]; s_first[2][t] = idx[2][0];
#endif
    }
    __syncthreads();
    const int c = t & (GATHER_GROUP - 1), grp = t / GATHER_GROUP;
    constexpr int NGRP = GATHER_BLOCK / GATHER_GROUP;
    const int cc = c < 5 ? c : 4;
    for (int it = 0; it < GATHER_GROUP; ++it) {
        const int al = it * NGRP + grp;
        float ph = 0.f, ex = 0.f, ey = 0.f, ez = 0.f;
#if QNEP_FIELD_BRICKS
        {
            // lane c owns corner (dx, dy, dz) of every brick: stencil slot o = 2 k + d - parity along each axis (weight 0 outside 0..4)
            const int dl[3] = {(c >> 2) & 1, (c >> 1) & 1, c & 1};
            const int hb[3] = {g.grid[0] >> 1, g.grid[1] >> 1, g.grid[2] >> 1};
            float wl[3][3];
            int bo[3][3];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int i0 = s_first[a][al], par = i0 & 1, b0 = i0 >> 1;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const int o = 2 * k + dl[a] - par;
                    wl[a][k] = (o >= 0 && o < 5) ? s_w[a][min(max(o, 0), 4)][al] : 0.f;
                    int bk = b0 + k;
                    bk = bk >= hb[a] ? bk - hb[a] : bk;
                    bo[a][k] = a == 0 ? bk * hb[1] * hb[2] : (a == 1 ? bk * hb[2] : bk);
                }
            }
            const float4* fc = field + c;
#pragma unroll
            for (int kx = 0; kx < 3; ++kx)
#pragma unroll
                for (int ky = 0; ky < 3; ++ky) {
                    const float wxy = wl[0][kx] * wl[1][ky];
                    const int oxy = bo[0][kx] + bo[1][ky];
#pragma unroll
                    for (int kz = 0; kz < 3; ++kz) {
                        const float w = wxy * wl[2][kz];
                        const float4 f = fc[(oxy + bo[2][kz]) << 3];
                        ph = fmaf(w, f.x, ph); ex = fmaf(w, f.y, ex);
                        ey = fmaf(w, f.z, ey); ez = fmaf(w, f.w, ez);
                    }
                }
        }
        if (false) {
#else
        if (c < 5) {
#endif
            const int zc = s_i[2][cc][al];
            float wy[5];
            int oy[5];
#pragma unroll
            for (int b = 0; b < 5; ++b) { wy[b] = s_w[1][b][al]; oy[b] = s_i[1][b][al] + zc; }
#pragma unroll
            for (int a = 0; a < 5; ++a) {
                const float wxa = s_w[0][a][al];
                const float4* row = field + s_i[0][a][al];
#pragma unroll
                for (int b = 0; b < 5; ++b) {
                    const float w = wxa * wy[b];
                    const float4 f = row[oy[b]];
                    ph = fmaf(w, f.x, ph); ex = fmaf(w, f.y, ex);
                    ey = fmaf(w, f.z, ey); ez = fmaf(w, f.w, ez);
                }
            }
            const float wzc = s_w[2][cc][al];
            ph *= wzc; ex *= wzc; ey *= wzc; ez *= wzc;
        }
#pragma unroll
        for (int o = GATHER_GROUP / 2; o > 0; o >>= 1) {
            ph += __shfl_xor_sync(0xffffffffu, ph, o);
            ex += __shfl_xor_sync(0xffffffffu, ex, o);
            ey += __shfl_xor_sync(0xffffffffu, ey, o);
            ez += __shfl_xor_sync(0xffffffffu, ez, o);
        }
        if (c == 0) { s_out[0][al] = ph; s_out[1][al] = ex; s_out[2][al] = ey; s_out[3][al] = ez; }
    }
    __syncthreads();
    if (p0 + t >= N) return;
    const int64_t p = cmi[p0 + t];                         // the block walked mesh-bin ranks; outputs in sorted order
    if (VMODE) {
        const float cw = (float)QNEP_K_COULOMB * q[p];     // Eq. 39
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const float v = cw * s_out[k][t];
            if (vr.row[k] >= 0) Wat[(int64_t)vr.row[k] * N + p] += v;
            if (vr.mirror[k] >= 0) Wat[(int64_t)vr.mirror[k] * N + p] += v;
        }
        return;
    }
    const float c2k = 2.f * (float)QNEP_K_COULOMB;
    phik[p] = c2k * s_out[0][t];                          // bracket of Eq. 38
    const float cq = -c2k * q[p];                         // Eq. 37
    float fx = cq * s_out[1][t], fy = cq * s_out[2][t], fz = cq * s_out[3][t];
    if (g.triclinic) {
        // the meshes carry the gradient along the reciprocal basis vectors (see KB): Cartesian F_a = sum_c hinv[3a + c] |h_c| f_c
        const float m0 = (float)g.L[0], m1 = (float)g.L[1], m2 = (float)g.L[2];
        const float f0 = fx * m0, f1 = fy * m1, f2 = fz * m2;
        fx = (float)g.hinv[0] * f0 + (float)g.hinv[1] * f1 + (float)g.hinv[2] * f2;
        fy = (float)g.hinv[3] * f0 + (float)g.hinv[4] * f1 + (float)g.hinv[5] * f2;
        fz = (float)g.hinv[6] * f0 + (float)g.hinv[7] * f1 + (float)g.hinv[8] * f2;
    }
    if (add_to_Fs) { Fs[p] += fx; Fs[N + p] += fy; Fs[2 * N + p] += fz; }
    else { Fs[p] = fx; Fs[N + p] = fy; Fs[2 * N + p] = fz; }
}

// ---- dispatch on the axis length ---------------------------------------------------------------------
template <typename F>
bool with_split(int n, F&& f)
{
    switch (n) {
        case 16: f(std::integral_constant<int, 4>(), std::integral_constant<int, 4>()); return true;
        case 32: f(std::integral_constant<int, 8>(), std::integral_constant<int, 4>()); return true;
        case 64: f(std::integral_constant<int, 8>(), std::integral_constant<int, 8>()); return true;
        case 128: f(std::integral_constant<int, 16>(), std::integral_constant<int, 8>()); return true;
        case 256: f(std::integral_constant<int, 16>(), std::integral_constant<int, 16>()); return true;
        case 512: f(std::integral_constant<int, 32>(), std::integral_constant<int, 16>()); return true;
    }
    return false;
}

template <typename K>
cudaError_t allow_smem(K kernel, size_t bytes)
{
    return bytes > 48 * 1024 ? cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) : cudaSuccess;
}

double alias_den(double z)
{
    const double z2 = z * z;   // Eq. 36 denominator polynomial (reading G2: -17/189)
    return 1.0 - 5.0 / 3.0 * z2 + 7.0 / 9.0 * z2 * z2 - 17.0 / 189.0 * z2 * z2 * z2 + 2.0 / 2835.0 * z2 * z2 * z2 * z2;
}

}  // namespace

// tables: twiddles and the separable factors of G^opt (Eq. 36)
int qnep_setup_pppm(qnep_handle* h)
{
    const int* grid = h->es.grid;
    for (int a = 0; a < 3; ++a) {
        const int n = grid[a];
        if (n < LINES || n > FFT_MAXN || (n & (n - 1))) { h->err = "PPPM grid must be a power of two in 16..512"; return QNEP_ERR_UNSUPPORTED; }
    }
    if (h->es.order != 5) { h->err = "PPPM order must be 5"; return QNEP_ERR_UNSUPPORTED; }
    const int64_t ng = (int64_t)grid[0] * grid[1] * grid[2];
    if (ng != h->ngrid) {
        cudaFree(h->d_mesh); cudaFree(h->d_cm1); cudaFree(h->d_cm2); cudaFree(h->d_field);
        cudaFree(h->d_cm3);      // allocated on demand by qnep_launch_pppm_atom_virial with the mesh size of that time
        h->d_mesh = nullptr; h->d_cm1 = nullptr; h->d_cm2 = nullptr; h->d_field = nullptr; h->d_cm3 = nullptr; h->cm3_ngrid = 0;
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_mesh, sizeof(float) * ng));
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_cm1, sizeof(float2) * ng));
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_cm2, sizeof(float2) * ng));
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_field, sizeof(float4) * ng));
        h->ngrid = ng;
    }
    {
        // half-spectrum array of the forward transform, [x][y][N2/2 + LINES]; the padding of the last tile stays zero
        const int64_t nh = grid[2] >= 2 * LINES ? (int64_t)grid[0] * grid[1] * (grid[2] / 2 + LINES) : 0;
        if (nh != h->nhalf) {
            cudaFree(h->d_half); h->d_half = nullptr;
            if (nh) QNEP_CUDA_OK(h, cudaMalloc(&h->d_half, sizeof(float2) * nh));
            h->nhalf = nh;
        }
        if (nh) QNEP_CUDA_OK(h, cudaMemset(h->d_half, 0, sizeof(float2) * nh));
    }
    if (!h->d_twiddle) QNEP_CUDA_OK(h, cudaMalloc(&h->d_twiddle, sizeof(float2) * 3 * FFT_MAXN));
    if (!h->d_gtab) QNEP_CUDA_OK(h, cudaMalloc(&h->d_gtab, sizeof(float) * 9 * FFT_MAXN));
    std::vector<float2> tw(3 * FFT_MAXN, make_float2(0.f, 0.f));
    std::vector<float> tab(9 * FFT_MAXN, 0.f);
    const double L[3] = {h->geo.L[0], h->geo.L[1], h->geo.L[2]};      // lengths of the cell vectors
    const bool tri = h->geo.triclinic != 0;
    for (int a = 0; a < 3; ++a) {
        const int n = grid[a];
        for (int t = 0; t < n; ++t) {
            const double ang = -2.0 * M_PI * t / n;
            tw[a * FFT_MAXN + t] = make_float2((float)cos(ang), (float)sin(ang));
        }
        for (int m = 0; m < n; ++m) {
            const int nn = m < n / 2 ? m : m - n;                 // -N/2 <= n < N/2 (:285)
            const double k = 2.0 * M_PI * nn / L[a];
            const double x = M_PI * nn / n;
            const double sc = x == 0.0 ? 1.0 : sin(x) / x;
            const double d = alias_den(sin(x));
            // triclinic: the Gaussian and k itself are formed per mesh point from the integer indices (see KB)
            tab[a * FFT_MAXN + m] = (float)((tri ? 1.0 : exp(-k * k / (4.0 * h->alpha * h->alpha))) * pow(sc, 10) / (d * d));
            tab[(3 + a) * FFT_MAXN + m] = tri ? (float)nn : (float)k;
            tab[(6 + a) * FFT_MAXN + m] = (2 * nn == -n) ? 0.f : (float)k;
        }
    }
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_twiddle, tw.data(), sizeof(float2) * 3 * FFT_MAXN, cudaMemcpyHostToDevice));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_gtab, tab.data(), sizeof(float) * 9 * FFT_MAXN, cudaMemcpyHostToDevice));
    return qnep_setup_sweep(h);
}

int qnep_launch_pppm(qnep_handle* h, bool virial, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 127) / 128);
    const int n0 = h->geo.grid[0], n1 = h->geo.grid[1], n2 = h->geo.grid[2];
    const float2* tw0 = h->d_twiddle;
    const float2* tw1 = h->d_twiddle + FFT_MAXN;
    const float2* tw2 = h->d_twiddle + 2 * FFT_MAXN;
    cudaError_t ce = cudaSuccess;
    auto note = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };

    // 1. spread: a shared-memory tile swept along x (pppm_sweep.cu), or one thread per atom for small systems
    const bool sweep = qnep_sweep_usable(h);
    if (sweep) {
        int rc = qnep_launch_spread_sweep(h, s);
        if (rc) return rc;
    } else {
        QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_mesh, 0, sizeof(float) * h->ngrid, s));
        k_spread<<<nb, 128, 0, s>>>(N, h->geo, h->d_mfrac, h->d_mi0, h->d_cm, h->d_q, h->d_mesh);
        h->launches += 1;
    }
    const Geometry& G = h->geo;
    const double vol = std::fabs(G.h[0] * (G.h[4] * G.h[8] - G.h[5] * G.h[7]) - G.h[1] * (G.h[3] * G.h[8] - G.h[5] * G.h[6]) +
                                 G.h[2] * (G.h[3] * G.h[7] - G.h[4] * G.h[6]));
    const float c0 = (float)(2.0 * M_PI / vol), inv4a2 = (float)(1.0 / (4.0 * h->alpha * h->alpha));
    const bool tri = G.triclinic != 0;
    KB kb;
    for (int k = 0; k < 9; ++k) kb.b[k] = (float)(2.0 * M_PI * G.hinv[k]);
    if (h->d_half) {
        // 2.-3. forward transform on the half spectrum (the mesh is real): z and y passes on [x][y][N2/2 + LINES],
        //       the fused x pass restores the full spectrum of M1, M2 on the way out
        const int NH = n2 / 2 + LINES;
        with_split(n2, [&](auto r1, auto r2) {
            constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
            using S = Split<R1, R2>;
            const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
            note(allow_smem(k_fft_z_fwd_half<R1, R2>, smem));
            k_fft_z_fwd_half<R1, R2><<<(unsigned)((int64_t)n0 * n1 / LINES), S::THREADS, smem, s>>>(h->d_mesh, h->d_half, tw2);
        });
        with_split(n1, [&](auto r1, auto r2) {
            constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
            using S = Split<R1, R2>;
            const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
            note(allow_smem(k_fft_strided<R1, R2, -1>, smem));
            k_fft_strided<R1, R2, -1><<<dim3((unsigned)((int64_t)n0 * NH / LINES), 1), S::THREADS, smem, s>>>(1, n0, n1, NH, h->d_half, h->d_half, tw1);
        });
        with_split(n0, [&](auto r1, auto r2) {
            constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
            using S = Split<R1, R2>;
            using SI = Split<R2, R1>;
            const size_t smem = sizeof(float2) * (LINES * (S::LP > SI::LP ? S::LP : SI::LP) + S::N) + sizeof(float) * 3 * S::N +
                                sizeof(float2) * S::E * S::THREADS;
            const unsigned nt = (unsigned)((int64_t)n1 * NH / LINES);
            auto go = [&](auto vf, auto tf) {
                constexpr bool V = decltype(vf)::value, TR = decltype(tf)::value;
                note(allow_smem(k_fft_x_fused_half<R1, R2, V, TR>, smem));
                k_fft_x_fused_half<R1, R2, V, TR><<<nt, S::THREADS, smem, s>>>(n0, n1, n2, h->d_half, h->d_cm1, h->d_cm2, tw0, h->d_gtab,
                                                                              h->d_gtab + 3 * FFT_MAXN, h->d_gtab + 6 * FFT_MAXN, c0, inv4a2, h->d_sums, kb);
            };
            if (virial) { if (tri) go(std::true_type(), std::true_type()); else go(std::true_type(), std::false_type()); }
            else { if (tri) go(std::false_type(), std::true_type()); else go(std::false_type(), std::false_type()); }
        });
    } else {
    // 2. forward z (real -> complex), forward y
    with_split(n2, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_z_fwd<R1, R2>, smem));
        k_fft_z_fwd<R1, R2><<<(unsigned)((int64_t)n0 * n1 / LINES), S::THREADS, smem, s>>>(h->d_mesh, h->d_cm1, tw2);
    });
    with_split(n1, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_strided<R1, R2, -1>, smem));
        k_fft_strided<R1, R2, -1><<<dim3((unsigned)((int64_t)n0 * n2 / LINES), 1), S::THREADS, smem, s>>>(1, n0, n1, n2, h->d_cm1, h->d_cm1, tw1);
    });
    // 3. + first inverse pass: x
    with_split(n0, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        using SI = Split<R2, R1>;
        const size_t smem = sizeof(float2) * (LINES * (S::LP > SI::LP ? S::LP : SI::LP) + S::N) + sizeof(float) * 3 * S::N;
        const unsigned nt = (unsigned)((int64_t)n1 * n2 / LINES);
        auto go = [&](auto vf, auto tf) {
            constexpr bool V = decltype(vf)::value, TR = decltype(tf)::value;
            note(allow_smem(k_fft_x_fused<R1, R2, V, TR>, smem));
            k_fft_x_fused<R1, R2, V, TR><<<nt, S::THREADS, smem, s>>>(n0, n1, n2, h->d_cm1, h->d_cm2, tw0, h->d_gtab, h->d_gtab + 3 * FFT_MAXN,
                                                                     h->d_gtab + 6 * FFT_MAXN, c0, inv4a2, h->d_sums, kb);
        };
        if (virial) { if (tri) go(std::true_type(), std::true_type()); else go(std::true_type(), std::false_type()); }
        else { if (tri) go(std::false_type(), std::true_type()); else go(std::false_type(), std::false_type()); }
    });
    }
    // 4. inverse y on both meshes, inverse z -> interleaved real fields
    with_split(n1, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_strided<R1, R2, +1>, smem));
        k_fft_strided<R1, R2, +1><<<dim3((unsigned)((int64_t)n0 * n2 / LINES), 2), S::THREADS, smem, s>>>(1, n0, n1, n2, h->d_cm1, h->d_cm2, tw1);
    });
    with_split(n2, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_z_fields<R1, R2>, smem));
        k_fft_z_fields<R1, R2><<<(unsigned)((int64_t)n0 * n1 / LINES), S::THREADS, smem, s>>>(h->d_cm1, h->d_cm2, h->d_field, tw2, n1);
    });
    // 5. gather
    const int nbg = (int)((N + GATHER_BLOCK - 1) / GATHER_BLOCK);
    k_gather<false><<<nbg, GATHER_BLOCK, 0, s>>>(N, h->geo, h->d_mfrac, h->d_mi0, h->d_cmi, h->d_q, h->d_field, h->model.mode == 1 ? 1 : 0, h->d_phik,
                                                 h->d_Fs, GatherRows(), nullptr);
    h->launches += 6;
    QNEP_CUDA_OK(h, ce);
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

// Per-atom virial of the reciprocal part (Eq. 39) into d_Wat [9][N], after qnep_launch_pppm of the same evaluation (the
// charge mesh is still in d_mesh; d_cm1, d_cm2 and d_field are free again).  A second forward transform on the FULL
// spectrum feeds the virial pass along x; the inverse y / z passes and the back-interpolation kernel are the ones of the
// main path, run on the three packed meshes.
int qnep_launch_pppm_atom_virial(qnep_handle* h, cudaStream_t s)
{
    const int64_t N = h->N;
    const int n0 = h->geo.grid[0], n1 = h->geo.grid[1], n2 = h->geo.grid[2];
    const float2* tw0 = h->d_twiddle;
    const float2* tw1 = h->d_twiddle + FFT_MAXN;
    const float2* tw2 = h->d_twiddle + 2 * FFT_MAXN;
    if (!h->d_cm3 || h->cm3_ngrid != h->ngrid) {         // first use, or the mesh changed size since (qnep_set_electrostatics)
        cudaFree(h->d_cm3); h->d_cm3 = nullptr; h->cm3_ngrid = 0;
        QNEP_CUDA_OK(h, cudaMalloc(&h->d_cm3, sizeof(float2) * h->ngrid));
        h->cm3_ngrid = h->ngrid;
    }
    cudaError_t ce = cudaSuccess;
    auto note = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
    const Geometry& G = h->geo;
    const double vol = std::fabs(G.h[0] * (G.h[4] * G.h[8] - G.h[5] * G.h[7]) - G.h[1] * (G.h[3] * G.h[8] - G.h[5] * G.h[6]) +
                                 G.h[2] * (G.h[3] * G.h[7] - G.h[4] * G.h[6]));
    const float c0 = (float)(2.0 * M_PI / vol), inv4a2 = (float)(1.0 / (4.0 * h->alpha * h->alpha));
    const bool tri = G.triclinic != 0;
    KB kb;
    for (int k = 0; k < 9; ++k) kb.b[k] = (float)(2.0 * M_PI * G.hinv[k]);
    with_split(n2, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_z_fwd<R1, R2>, smem));
        k_fft_z_fwd<R1, R2><<<(unsigned)((int64_t)n0 * n1 / LINES), S::THREADS, smem, s>>>(h->d_mesh, h->d_cm3, tw2);
    });
    with_split(n1, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_strided<R1, R2, -1>, smem));
        k_fft_strided<R1, R2, -1><<<dim3((unsigned)((int64_t)n0 * n2 / LINES), 1), S::THREADS, smem, s>>>(1, n0, n1, n2, h->d_cm3, h->d_cm3, tw1);
    });
    with_split(n0, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        using SI = Split<R2, R1>;
        const size_t smem = sizeof(float2) * (LINES * (S::LP > SI::LP ? S::LP : SI::LP) + S::N) + sizeof(float) * 2 * S::N;
        if (tri) {
            note(allow_smem(k_fft_x_virial<R1, R2, true>, smem));
            k_fft_x_virial<R1, R2, true><<<(unsigned)((int64_t)n1 * n2 / LINES), S::THREADS, smem, s>>>(n0, n1, n2, h->d_cm1, h->d_cm2, h->d_cm3, tw0, h->d_gtab,
                                                                                                       h->d_gtab + 3 * FFT_MAXN, c0, inv4a2, kb);
        } else {
            note(allow_smem(k_fft_x_virial<R1, R2, false>, smem));
            k_fft_x_virial<R1, R2, false><<<(unsigned)((int64_t)n1 * n2 / LINES), S::THREADS, smem, s>>>(n0, n1, n2, h->d_cm1, h->d_cm2, h->d_cm3, tw0, h->d_gtab,
                                                                                                        h->d_gtab + 3 * FFT_MAXN, c0, inv4a2, kb);
        }
    });
    with_split(n1, [&](auto r1, auto r2) {
        constexpr int R1 = decltype(r1)::value, R2 = decltype(r2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_strided<R1, R2, +1>, smem));
        k_fft_strided<R1, R2, +1><<<dim3((unsigned)((int64_t)n0 * n2 / LINES), 2), S::THREADS, smem, s>>>(1, n0, n1, n2, h->d_cm1, h->d_cm2, tw1);
        k_fft_strided<R1, R2, +1><<<dim3((unsigned)((int64_t)n0 * n2 / LINES), 1), S::THREADS, smem, s>>>(1, n0, n1, n2, h->d_cm3, h->d_cm3, tw1);
    });
    const int nbg = (int)((N + GATHER_BLOCK - 1) / GATHER_BLOCK);
    if (h->model.mode != 1) QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_Wat, 0, sizeof(float) * 9 * N, s));     // mode 1: k_realspace wrote d_Wat
    GatherRows r1 = {{0, 4, 8, 1}, {-1, -1, -1, 3}};      // (W_xx, W_yy, W_zz, W_xy)
    GatherRows r2 = {{2, 5, -1, -1}, {6, 7, -1, -1}};     // (W_xz, W_yz, W_xz, W_yz): the second copy is not used
    with_split(n2, [&](auto q1, auto q2) {
        constexpr int R1 = decltype(q1)::value, R2 = decltype(q2)::value;
        using S = Split<R1, R2>;
        const size_t smem = sizeof(float2) * (LINES * S::LP + S::N);
        note(allow_smem(k_fft_z_fields<R1, R2>, smem));
        k_fft_z_fields<R1, R2><<<(unsigned)((int64_t)n0 * n1 / LINES), S::THREADS, smem, s>>>(h->d_cm1, h->d_cm2, h->d_field, tw2, n1);
        k_gather<true><<<nbg, GATHER_BLOCK, 0, s>>>(N, h->geo, h->d_mfrac, h->d_mi0, h->d_cmi, h->d_q, h->d_field, 0, nullptr, nullptr, r1, h->d_Wat);
        k_fft_z_fields<R1, R2><<<(unsigned)((int64_t)n0 * n1 / LINES), S::THREADS, smem, s>>>(h->d_cm3, h->d_cm3, h->d_field, tw2, n1);
        k_gather<true><<<nbg, GATHER_BLOCK, 0, s>>>(N, h->geo, h->d_mfrac, h->d_mi0, h->d_cmi, h->d_q, h->d_field, 0, nullptr, nullptr, r2, h->d_Wat);
    });
    h->launches += 9;
    QNEP_CUDA_OK(h, ce);
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}
