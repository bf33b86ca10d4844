// fft_reg.cuh -- register-resident small FFTs for the hand-written 3-D FFT of pppm.cu (PAPER.md :302
// names the transforms; reading S11: both directions unnormalised, forward e^{-i...}, inverse e^{+i...}).
//
// A line of length N = R1 * R2 is transformed by the Cooley-Tukey split  n = t + R2 m  ->  k = k2 + R1 k1:
//   stage 1: R1-point DFT over m for each residue t              (in registers)
//   twiddle: omega_N^{t k2}
//   exchange through shared memory (the only data movement between threads)
//   stage 2: R2-point DFT over t for each k2                     (in registers)
// Every index below is a compile-time constant after unrolling, so the small DFTs compile to straight-line
// FADD/FMUL/FFMA code on registers with immediate twiddles.
#pragma once
#include <cuda_runtime.h>

#include <type_traits>

namespace fftreg {

#ifdef __CUDACC__
#define FFT_HD __host__ __device__ __forceinline__
#else
#define FFT_HD inline
#endif

// cos(2 pi k / 32); nested selects (no table) so that it folds to an immediate once k is a constant
FFT_HD constexpr float cos32_oct(int k)      // k = 0..8
{
    return k == 0 ? 1.0f : k == 1 ? 0.98078528040323043f : k == 2 ? 0.92387953251128674f : k == 3 ? 0.83146961230254524f :
           k == 4 ? 0.70710678118654752f : k == 5 ? 0.55557023301960218f : k == 6 ? 0.38268343236508977f :
           k == 7 ? 0.19509032201612825f : 0.0f;
}
FFT_HD constexpr float cos32(int k)
{
    k &= 31;
    if (k > 16) k = 32 - k;          // cos is even
    return k <= 8 ? cos32_oct(k) : -cos32_oct(16 - k);
}
FFT_HD constexpr float sin32(int k) { return cos32(k - 8); }

FFT_HD constexpr int bitrev(int x, int bits)
{
    int r = 0;
    for (int i = 0; i < bits; ++i) r |= ((x >> i) & 1) << (bits - 1 - i);
    return r;
}
FFT_HD constexpr int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

// compile-time loop: f(integral_constant<int, B>), ..., f(integral_constant<int, E - 1>) -- no loop is left for the
// unroller to refuse, so every register index and twiddle below is a constant expression
template <int B, int E, typename F>
FFT_HD void static_for(F&& f)
{
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// in-place R-point DFT of v[0..R-1] (stride 1), natural order in and out; SIGN = -1 forward, +1 inverse
template <int R, int SIGN>
FFT_HD void dft(float2* v)
{
    static_assert(R == 2 || R == 4 || R == 8 || R == 16 || R == 32, "radix");
    constexpr int LOG = ilog2(R);
    // bit-reversal permutation (compile-time swaps)
    static_for<0, R>([&](auto ic) {
        constexpr int i = decltype(ic)::value;
        constexpr int j = bitrev(i, LOG);
        if constexpr (j > i) { const float2 tmp = v[i]; v[i] = v[j]; v[j] = tmp; }
    });
    // decimation in time
    static_for<0, LOG>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        constexpr int half = 1 << s, len = half << 1;
        static_for<0, R / 2>([&](auto bc) {
            constexpr int idx = decltype(bc)::value;
            constexpr int base = (idx / half) * len, j = idx % half;
            constexpr int tw = j * (32 / len);            // omega_len^j = omega_32^tw
            const float2 a = v[base + j];
            float2 b = v[base + j + half];
            if constexpr (tw == 0) {
            } else if constexpr (tw == 8) {               // multiply by SIGN * i
                b = SIGN < 0 ? make_float2(b.y, -b.x) : make_float2(-b.y, b.x);
            } else {
                constexpr float c = cos32(tw), sgn = SIGN < 0 ? -sin32(tw) : sin32(tw);
                b = make_float2(b.x * c - b.y * sgn, b.x * sgn + b.y * c);
            }
            v[base + j] = make_float2(a.x + b.x, a.y + b.y);
            v[base + j + half] = make_float2(a.x - b.x, a.y - b.y);
        });
    });
}

}  // namespace fftreg
