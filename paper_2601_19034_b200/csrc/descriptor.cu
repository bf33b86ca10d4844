// descriptor.cu -- steps a2, a3, a4, a5, a10, a11, a12 of SURVEY.md 8(a):
//   radial / angular NEP descriptors (PAPER.md :56; readings S1-S3),
//   the per-atom network with the extra charge output (Eq. 1, :58-60),
//   Eq. 33 neutralisation, the folded back-propagation  Fp = dU_i/dD + phi_eff dq_i/dD  (:140, Eq. 14, 17),
//   partial forces, force / virial assembly (Eq. 11, 12) and the Born effective charges (Eq. 28).
//
// One thread owns one atom; atoms are (type, cell)-sorted so a warp is type-uniform and its
// neighbour gathers hit the same cache lines.  All per-neighbour state lives in registers.
//
// Per step the skin list is walked ONCE (k_pairs): it accumulates the radial descriptors and emits the
// exact lists of this step -- the live radial list (packed indices) and the live angular pairs
// (dx, dy, dz, j | tj), which the angular kernels then stream coalesced, with no gather and no skin-shell
// divergence.
//
// Algebra used to keep the hot loops on the FP32 FMA pipe:
//   * radial:  D_n = sum_j sum_k c^{ti tj}_{nk} f_k(r_ij) = sum_t sum_k c^{ti t}_{nk} S^t_k,
//     S^t_k = sum_{j in t} f_k(r_ij): the per-neighbour work is the 9 basis values only; the
//     coefficient contraction is done once per atom.  Backward likewise with
//     P^{t}_k = sum_n Fp_n c^{ti t}_{nk}.
//   * angular: A_nlm = sum_j g_n(r_ij) b_lm(rhat_ij) with 24 real harmonic polynomials b_lm;
//     D_nl = sum_m C_lm A_nlm^2 equals the Legendre double sum of the definition by the addition
//     theorem (weights C_lm are exact rationals, see harmonic weights below).
//   * F_ji of the radial part is recomputed by atom i from P^{ti}_k of atom j (no atomics, no
//     pair storage); the angular F_ij is added to atom i's own sum and scattered to atom j with
//     fp32 atomic adds (RED) into a zeroed accumulator.
#include "qnep_internal.cuh"

#include <algorithm>
#include <type_traits>

namespace {

constexpr int NB = QNEP_NB;       // 9 basis functions
constexpr int NR = QNEP_NRAD;     // 5 radial functions
constexpr int KP = QNEP_KPAD;     // padded row
constexpr int NLM = QNEP_NLM;
constexpr int ND = QNEP_NDESC;

// addition-theorem weights: P_l(u.v) = sum_m C_lm b_lm(u) b_lm(v)
__constant__ float c_Clm[NLM] = {1.f, 1.f, 1.f,
                                 0.25f, 3.f, 3.f, 0.75f, 0.75f,
                                 0.25f, 0.375f, 0.375f, 3.75f, 3.75f, 0.625f, 0.625f,
                                 1.f / 64.f, 0.625f, 0.625f, 0.3125f, 0.3125f, 4.375f, 4.375f, 35.f / 64.f, 35.f / 64.f};
__host__ __device__ __forceinline__ constexpr int l_of_lm(int lm) { return lm < 3 ? 0 : (lm < 8 ? 1 : (lm < 15 ? 2 : 3)); }

// f_k(r) = 1/2 [T_k(x) + 1] f_c(r), x = 2 (r/rc - 1)^2 - 1, f_c = 1/2 [1 + cos(pi r / rc)]   (S1)
template <bool VAL, bool DERIV>
__device__ __forceinline__ void cheb_basis(float r, float rcinv, float* __restrict__ f, float* __restrict__ df)
{
    const float t = r * rcinv;
    float sn, cs;                                   // MUFU sin / cos of pi t, t in [0, 1]: abs error < 5e-7
    if (DERIV) __sincosf(3.14159265358979f * t, &sn, &cs);
    else cs = __cosf(3.14159265358979f * t);
    const float fc = 0.5f + 0.5f * cs;
    const float tm1 = t - 1.f;
    const float x = 2.f * tm1 * tm1 - 1.f;
    const float hfc = 0.5f * fc;
    float dfc = 0.f, dx = 0.f, hdxfc = 0.f, hdfc = 0.f;
    if (DERIV) {
        dfc = -1.5707963267948966f * rcinv * sn;
        dx = 4.f * tm1 * rcinv;
        hdxfc = 0.5f * dx * fc;
        hdfc = 0.5f * dfc;
    }
    float Tm = 1.f, Tc = x, dTm = 0.f, dTc = 1.f;
    if (VAL) { f[0] = fc; f[1] = hfc * (x + 1.f); }
    if (DERIV) { df[0] = dfc; df[1] = hdxfc + hdfc * (x + 1.f); }
#pragma unroll
    for (int k = 2; k < NB; ++k) {
        const float Tn = 2.f * x * Tc - Tm;
        if (VAL) f[k] = hfc * (Tn + 1.f);
        if (DERIV) {
            const float dTn = 2.f * Tc + 2.f * x * dTc - dTm;
            df[k] = hdxfc * dTn + hdfc * (Tn + 1.f);
            dTm = dTc; dTc = dTn;
        }
        Tm = Tc; Tc = Tn;
    }
}

// Derivative basis in the form used by the radial force kernel:  f_k'(r) = A k U_{k-1}(x) + B (T_k(x) + 1)  with
// A = 1/2 fc dx/dr, B = 1/2 dfc/dr (T_k' = k U_{k-1}; f_0 = fc = 1/2 fc (T_0 + 1) fits the same formula), so
//   sum_k a_k f_k'(r) = A sum_{k>=1} a_k kU_k + B sum_k a_k Tp_k,   kU_k = k U_{k-1},  Tp_k = T_k + 1.
struct ChebDeriv {
    float A, B, hfc;  // hfc = 1/2 fc(r)
    float kU[NB];     // kU[0] = 0 (unused)
    float Tp[NB];
    __device__ __forceinline__ void eval(float r, float rcinv)
    {
        const float t = r * rcinv;
        float sn, cs;
        __sincosf(3.14159265358979f * t, &sn, &cs);
        const float tm1 = t - 1.f;
        const float x = 2.f * tm1 * tm1 - 1.f, x2 = x + x;
        hfc = 0.25f + 0.25f * cs;
        A = hfc * (4.f * tm1 * rcinv);                           // 1/2 fc dx/dr, x = 2 (t - 1)^2 - 1
        B = -0.7853981633974483f * rcinv * sn;                   // 1/2 * (-pi / (2 rc)) sin(pi t)
        float Tm = 1.f, Tc = x, Um = 1.f, Uc = x2;               // T_0, T_1, U_0, U_1
        Tp[0] = 2.f; Tp[1] = x + 1.f;
        kU[0] = 0.f; kU[1] = 1.f; kU[2] = 2.f * Uc;
#pragma unroll
        for (int k = 2; k < NB; ++k) {
            const float Tn = fmaf(x2, Tc, -Tm);
            Tp[k] = Tn + 1.f;
            Tm = Tc; Tc = Tn;
            if (k + 1 < NB) {
                const float Un = fmaf(x2, Uc, -Um);              // U_k
                kU[k + 1] = (float)(k + 1) * Un;
                Um = Uc; Uc = Un;
            }
        }
    }
    __device__ __forceinline__ float dot(const float (&a)[NB]) const
    {
        float du = a[1], dt = a[0] * Tp[0];
#pragma unroll
        for (int k = 1; k < NB; ++k) dt = fmaf(a[k], Tp[k], dt);
#pragma unroll
        for (int k = 2; k < NB; ++k) du = fmaf(a[k], kU[k], du);
        return fmaf(A, du, B * dt);
    }
    // the same contraction with a_1..a_8 given as four register pairs (a_1, a_2) .. (a_7, a_8): packed FMAs
    __device__ __forceinline__ float dot_pairs(float a0, const float2 (&ap)[4]) const
    {
        float2 dt = __fmul2_rn(ap[0], make_float2(Tp[1], Tp[2])), du = __fmul2_rn(ap[0], make_float2(1.f, kU[2]));
#pragma unroll
        for (int m = 1; m < 4; ++m) {
            dt = __ffma2_rn(ap[m], make_float2(Tp[2 * m + 1], Tp[2 * m + 2]), dt);
            du = __ffma2_rn(ap[m], make_float2(kU[2 * m + 1], kU[2 * m + 2]), du);
        }
        return fmaf(A, du.x + du.y, B * fmaf(a0, Tp[0], dt.x + dt.y));
    }
};

// MUFU.RSQ without the denormal range fix-up of rsqrtf (arguments here are squared distances >= 1e-12)
__device__ __forceinline__ float fast_rsqrt(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ double block_sum(double v, double* sh)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = lane < (blockDim.x >> 5) ? sh[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
    }
    return r;   // valid in thread 0
}

// ------------------------------------------------------------------------------------------
// asynchronous global -> shared copies (LDGSTS): a thread streams its own list rows through a small ring in
// shared memory, so many loads are in flight per thread at no register cost.  A thread only ever reads what it
// copied itself, so cp.async.wait_group is the only synchronisation needed.  (Used for streams only: LDGSTS does
// not allocate in L1, so gathers that profit from L1 hits use plain loads into register rotations instead.)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void cp_async16_cg(void* sm, const void* g)      // streams: bypass L1
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(sm)), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory"); }

// ------------------------------------------------------------------------------------------
// a2: one walk over the skin list: the exact lists of this step and the radial descriptors
//   live radial entry : the skin-list word (sorted index | cell offset of the image << 26), type-major like the skin list
//                       (warp-tiled int4 layout); lvRend[t][p] = end of the species-t segment
//   live angular pair : (dx, dy, dz, bits(sorted index | type << 26: QNEP_NL_SHIFT; index limit 2^26))
// The kernel is bound by L1 wavefronts (gathers of 16 bytes from ~15 lines per warp instruction, the queue and the
// shift table in shared memory) and by issue slots, so both phases are kept to the instructions they need:
//   phase 1, per SKIN entry (all lanes busy): list word -> position gather -> distance test; accepted entries are
//     pushed to a per-thread RING in shared memory (word, r^2) and, inside the angular cutoff, appended to the
//     angular pair list.  Bounds, prefetch and species are decided once per list vector: the build pads every species
//     segment to a multiple of four slots (k_build_lists), nlRend[t][p] holds the segment ends.
//   phase 2, per ACCEPTED entry, four at a time (one int4 of the live radial list): basis functions f_k(r) and
//     S^t_k += f_k.  After every round of PAIRS_CH slots a warp pops the SAME number of entries from all its rings
//     (what the emptiest lane has, but at least what the fullest lane must give up to leave room for the next
//     round), so the binomial scatter of the acceptance count over a round does not idle lanes; what stays in a
//     ring waits for the next round, the last round drains.
// ------------------------------------------------------------------------------------------
constexpr int PAIRS_BLOCK = 128;
constexpr int PAIRS_CH = 16;                 // skin slots per round (four list vectors)
constexpr int PAIRS_QCAP = 2 * PAIRS_CH;     // ring capacity per thread
constexpr int PAIRS_LD = 8;                  // list vectors in flight per thread (power of two)
constexpr size_t PAIRS_SMEM = sizeof(int4) * PAIRS_LD * PAIRS_BLOCK + sizeof(int) * 2 * PAIRS_QCAP * PAIRS_BLOCK;

__device__ __forceinline__ int4 ldg_stream(const int4* p)        // streamed once: do not allocate in L1
{
    int4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ int word_of(const int4& v, int u) { return u == 0 ? v.x : (u == 1 ? v.y : (u == 2 ? v.z : v.w)); }
// position gather: one LOP3 + one IMAD.WIDE for the address (the compiler's own sequence re-reads the base pointer from
// the constant bank and adds with carry: five instructions per gather)
__device__ __forceinline__ float4 gather_pos(const float4* __restrict__ base, int word)
{
    const unsigned idx = (unsigned)word & QNEP_NL_MASK;
    unsigned long long a;
    asm("mad.wide.u32 %0, %1, 16, %2;" : "=l"(a) : "r"(idx), "l"(base));
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(a));
    return v;
}
__device__ __forceinline__ void sts_pair(unsigned addr, int w, float r2, int second_offset_bytes)
{
    asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(w) : "memory");
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr + second_offset_bytes), "f"(r2) : "memory");
}
// store of row `row` of a warp-tiled float4 list (rows are QNEP_TILE float4 = 512 bytes apart): one IMAD.WIDE + STG
__device__ __forceinline__ void stg_tiled_row(float4* base, int row, float x, float y, float z, int w)
{
    unsigned long long a;
    asm("mad.wide.u32 %0, %1, 512, %2;" : "=l"(a) : "r"((unsigned)row), "l"(base));
    asm volatile("st.global.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(a), "f"(x), "f"(y), "f"(z), "f"(__int_as_float(w)) : "memory");
}
__device__ __forceinline__ int lds_b32(unsigned addr) { int v; asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); return v; }
__device__ __forceinline__ float lds_f32(unsigned addr) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory"); return v; }

template <int T, bool TRI>
__global__ void __launch_bounds__(PAIRS_BLOCK)
k_pairs(int64_t N, Geometry g, const float4* __restrict__ xyzt, const int4* __restrict__ nl,
        const int* __restrict__ nn, const int* __restrict__ nlRend, const float* __restrict__ cR, float rcinv, int capR, int capLR, int capLA,
        int4* __restrict__ lvR, int* __restrict__ nlvR, int* __restrict__ lvRend,
        float4* __restrict__ lvA, int* __restrict__ nlvA, float* __restrict__ D, int* __restrict__ flags)
{
    static_assert(PAIRS_CH == 16 && (PAIRS_QCAP & (PAIRS_QCAP - 1)) == 0, "four list vectors per round, power-of-two ring");
    __shared__ float sh_c[T * T * NR * KP];
    extern __shared__ __align__(16) unsigned char sh_dyn[];  // PAIRS_SMEM bytes (beyond the 48 KB of static shared memory)
    int4 (*sh_l)[PAIRS_BLOCK] = reinterpret_cast<int4 (*)[PAIRS_BLOCK]>(sh_dyn);                                      // [PAIRS_LD]: list vectors in flight
    int (*sh_q)[PAIRS_QCAP][PAIRS_BLOCK] = reinterpret_cast<int (*)[PAIRS_QCAP][PAIRS_BLOCK]>(sh_dyn + sizeof(int4) * PAIRS_LD * PAIRS_BLOCK);   // [2]: ring of words, then r^2 (as bits)
    constexpr int QROW = PAIRS_BLOCK * 4, QR2 = PAIRS_QCAP * QROW, QMASK = QR2 - 1;   // bytes per slot, offset of the r^2 half, ring wrap
    for (int i = threadIdx.x; i < T * T * NR * KP; i += blockDim.x) sh_c[i] = cR[i];
    __syncthreads();
    const CellVecs cv = qnep_cell_vecs(g.cellv, TRI ? 1 : 0);      // compile-time switch: the orthorhombic walk pays nothing for the general cell
    const int tid = threadIdx.x;
    const int64_t p0 = blockIdx.x * (int64_t)blockDim.x + tid;
    const bool live = p0 < N;                                // threads beyond N stay for the warp votes, with an empty list
    const int64_t p = live ? p0 : N - 1;
    const float4 xi = xyzt[p];
    const int ti = __float_as_int(xi.w);
    const int n4 = live ? (nn[p] >> 2) : 0;                  // list vectors (the count is a multiple of four)
    int segend[T], acc_end[T];                               // skin slot / accepted count at which species t ends
#pragma unroll
    for (int t = 0; t < T; ++t) { segend[t] = (t < T - 1 && live) ? nlRend[(int64_t)t * N + p] : 0x7fffffff; acc_end[t] = 0x7fffffff; }
    const int4* lbase = nl + qnep_tiled_base(p, capR / 4);
    // List vectors come through a cp.async ring PAIRS_LD vectors deep in shared memory (they stream from DRAM); vector
    // gv + 2 is taken from the ring into registers at the top of iteration gv and feeds the position gathers at once
    // (eight slots ahead: the gathers mostly come from L2), lv[gv & 3] holds the vector being processed.  Beyond the
    // end the registers hold the atom itself, so the gathers need no bound check.
    const int4 filler = make_int4((int)p, (int)p, (int)p, (int)p);
#pragma unroll
    for (int k = 0; k < PAIRS_LD; ++k) {
        if (k < n4) cp_async16_cg(&sh_l[k][tid], lbase + (int64_t)k * QNEP_TILE);
        cp_async_commit();
    }
    cp_async_wait<PAIRS_LD - 2>();
    int4 lv[4];
    lv[0] = 0 < n4 ? sh_l[0][tid] : filler;
    lv[1] = 1 < n4 ? sh_l[1][tid] : filler;
    lv[2] = filler; lv[3] = filler;
#pragma unroll
    for (int k = 0; k < 2; ++k) {                            // slots 0 and 1 are free again: vectors PAIRS_LD, PAIRS_LD + 1
        if (PAIRS_LD + k < n4) cp_async16_cg(&sh_l[k][tid], lbase + (int64_t)(PAIRS_LD + k) * QNEP_TILE);
        cp_async_commit();
    }
    float4 ring[8];                                          // ring[4 (gv & 1) + u] holds the position of the atom of slot 4 gv + u
#pragma unroll
    for (int u = 0; u < 8; ++u) ring[u] = gather_pos(xyzt, word_of(lv[u >> 2], u & 3));
    float S[T][NB];                                          // S^t_k without the "+1" part: sum_j 1/2 fc T_k
    float S1[T];                                             // sum_j 1/2 fc
#pragma unroll
    for (int t = 0; t < T; ++t) {
        S1[t] = 0.f;
#pragma unroll
        for (int k = 0; k < NB; ++k) S[t][k] = 0.f;
    }
    int cA_ = 0, head = 0, tail = 0;                         // angular pairs; accepted entries consumed / produced
    int4* outR = lvR + qnep_tiled_base(p, capLR / 4);
    float4* outA = lvA + qnep_tiled_base(p, capLA);
    const unsigned qbase = (unsigned)__cvta_generic_to_shared(&sh_q[0][0][tid]);
    unsigned qoff = 0;                                       // byte offset of the ring slot of accepted entry `tail`
    const int nround = __reduce_max_sync(0xffffffffu, (n4 + 3) >> 2);
    for (int c = 0; c < nround; ++c) {
        // ---- phase 1 ----
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const int gv = 4 * c + v;
            // vector gv + 2 from the ring; its slot is refilled with vector gv + 2 + PAIRS_LD
            cp_async_wait<PAIRS_LD - 1>();                   // groups issued so far: PAIRS_LD + 2 + gv, one per vector; vector gv + 2 has landed
            lv[(v + 2) & 3] = gv + 2 < n4 ? sh_l[(gv + 2) & (PAIRS_LD - 1)][tid] : filler;
            if (gv + 2 + PAIRS_LD < n4) cp_async16_cg(&sh_l[(gv + 2) & (PAIRS_LD - 1)][tid], lbase + (int64_t)(gv + 2 + PAIRS_LD) * QNEP_TILE);
            cp_async_commit();
            float4 xjv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                xjv[u] = ring[4 * (v & 1) + u];
                ring[4 * (v & 1) + u] = gather_pos(xyzt, word_of(lv[(v + 2) & 3], u));
            }
            int tjv = 0;
#pragma unroll
            for (int t = 0; t < T - 1; ++t) {
                if (4 * gv == segend[t]) acc_end[t] = tail;
                tjv += (4 * gv >= segend[t]) ? 1 : 0;
            }
            const int tjbits = tjv << QNEP_NL_SHIFT;
            const bool act = gv < n4;
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int e = word_of(lv[v & 3], u);
                const float4 xj = xjv[u];
                float dx = xj.x - xi.x, dy = xj.y - xi.y, dz = xj.z - xi.z;
                qnep_add_image_shift(e, cv, dx, dy, dz);
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                if (act && r2 < g.rc_r2 && r2 >= 1e-12f) {
                    sts_pair(qbase + qoff, e, r2, QR2);
                    qoff = (qoff + QROW) & QMASK;
                    ++tail;
                    if (r2 < g.rc_a2) {
                        if (cA_ < capLA) stg_tiled_row(outA, cA_, dx, dy, dz, (e & QNEP_NL_MASK) | tjbits);
                        ++cA_;
                    }
                }
            }
        }
        // ---- phase 2 ----
        const int fill = tail - head;
        const bool last = c == nround - 1;
        const int mn = __reduce_min_sync(0xffffffffu, fill), mx = __reduce_max_sync(0xffffffffu, fill);
        const int npop = last ? ((mx + 3) & ~3) : max(mn & ~3, (mx - PAIRS_CH + 3) & ~3);
        const int mine = last ? fill : (min(npop, fill) & ~3);
        for (int k = 0; k < npop; k += 4) {
            if (k < mine) {
                int w4[4];
                const unsigned qa = qbase + (unsigned)((head + k) & (PAIRS_QCAP - 1)) * QROW;   // head + k is a multiple of four: no wrap inside the group
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int gidx = head + k + u;                                   // accepted entry number gidx of this atom
                    const bool valid = k + u < mine;                                 // false only in the tail of the last round
                    const float r2 = valid ? lds_f32(qa + u * QROW + QR2) : 1.f;
                    w4[u] = valid ? lds_b32(qa + u * QROW) : QNEP_NL_EMPTY;
                    // 1/2 fc(r) T_k(x), k = 0..8   (f_k = 1/2 fc (T_k + 1): the "+1" part is accumulated once in S1)
                    const float tt = r2 * fast_rsqrt(r2) * rcinv;
                    const float hfc = valid ? 0.25f + 0.25f * __cosf(3.14159265358979f * tt) : 0.f;
                    const float tm1 = tt - 1.f;
                    const float x = 2.f * tm1 * tm1 - 1.f, x2 = x + x;
                    float a[T];
#pragma unroll
                    for (int t = 0; t < T; ++t) a[t] = (T == 1 || ((t == 0 || gidx >= acc_end[t - 1]) && (t == T - 1 || gidx < acc_end[t]))) ? hfc : 0.f;
                    float Tm = 1.f, Tc = x;
#pragma unroll
                    for (int t = 0; t < T; ++t) { S1[t] += a[t]; S[t][1] = fmaf(a[t], Tc, S[t][1]); }
#pragma unroll
                    for (int kk = 2; kk < NB; ++kk) {
                        const float Tn = fmaf(x2, Tc, -Tm);
#pragma unroll
                        for (int t = 0; t < T; ++t) S[t][kk] = fmaf(a[t], Tn, S[t][kk]);
                        Tm = Tc; Tc = Tn;
                    }
                }
                if (head + k < capLR) outR[(int64_t)((head + k) >> 2) * QNEP_TILE] = make_int4(w4[0], w4[1], w4[2], w4[3]);
            }
        }
        head += mine;
    }
    if (!live) return;
    nlvR[p] = min(tail, capLR);
    nlvA[p] = min(cA_, capLA);
#pragma unroll
    for (int t = 0; t < T; ++t) lvRend[(int64_t)t * N + p] = min(t < T - 1 ? min(acc_end[t], tail) : tail, capLR);
    if (tail > capLR) atomicMax(&flags[FLAG_MAX_LR], tail);
    if (cA_ > capLA) atomicMax(&flags[FLAG_MAX_LA], cA_);
    // f_0 = fc = 2 (1/2 fc): S^t_0 = 2 S1;  f_k = 1/2 fc T_k + 1/2 fc: S^t_k = S[t][k] + S1
#pragma unroll
    for (int nidx = 0; nidx < NR; ++nidx) {
        float d = 0.f;
#pragma unroll
        for (int t = 0; t < T; ++t) {
            const float* c = sh_c + ((ti * T + t) * NR + nidx) * KP;
            d = fmaf(c[0], 2.f * S1[t], d);
#pragma unroll
            for (int k = 1; k < NB; ++k) d = fmaf(c[k], S[t][k] + S1[t], d);
        }
        D[(int64_t)nidx * N + p] = d;
    }
}

// ------------------------------------------------------------------------------------------
// real harmonic polynomials b_lm(u), l = 1..4 (unit vector u = (x, y, z))
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void harmonics(float x, float y, float z, float* __restrict__ b)
{
    const float x2 = x * x, y2 = y * y, z2 = z * z, xy = x * y;
    const float x2my2 = x2 - y2;
    b[0] = z; b[1] = x; b[2] = y;
    b[3] = 3.f * z2 - 1.f; b[4] = x * z; b[5] = y * z; b[6] = x2my2; b[7] = 2.f * xy;
    const float f5 = 5.f * z2 - 1.f;
    b[8] = (5.f * z2 - 3.f) * z; b[9] = f5 * x; b[10] = f5 * y; b[11] = x2my2 * z; b[12] = 2.f * xy * z;
    b[13] = (x2 - 3.f * y2) * x; b[14] = (3.f * x2 - y2) * y;
    const float f7 = 7.f * z2 - 1.f, f73 = 7.f * z2 - 3.f;
    b[15] = (35.f * z2 - 30.f) * z2 + 3.f; b[16] = f73 * x * z; b[17] = f73 * y * z; b[18] = f7 * x2my2;
    b[19] = f7 * 2.f * xy; b[20] = (x2 - 3.f * y2) * x * z; b[21] = (3.f * x2 - y2) * y * z;
    b[22] = x2my2 * x2my2 - 4.f * x2 * y2; b[23] = 4.f * x2my2 * xy;
}

// ------------------------------------------------------------------------------------------
// a3: angular descriptors; A_nlm kept for the backward pass
// ------------------------------------------------------------------------------------------
// The live angular pairs are streamed through a cp.async ring ANG_DEPTH rows deep (the kernels hold 120+ accumulators
// in registers, so occupancy is low and the loads must be issued far ahead).
constexpr int ANG_BLOCK = 64, ANG_DEPTH = 8;
constexpr int FA_KP2 = 10;     // float2 per row of the packed coefficient table of k_force_angular

// NEP4's higher-body terms of one radial channel (reading Z2) from the real-harmonic sums A_lm, lm = 0..7
// (b_0..2 = z, x, y; b_3..7 = 3z^2 - 1, xz, yz, x^2 - y^2, 2xy): the l = 1 vector w = sum_j g rhat and the traceless l = 2
// tensor T = sum_j g (rhat rhat^T - 1/3), stored as (xx, yy, zz, xy, xz, yz); S = T^2.
__device__ __forceinline__ void hb_moments(const float (&A)[8], float (&Tn)[6], float (&Sn)[6], float& w2)
{
    w2 = A[0] * A[0] + A[1] * A[1] + A[2] * A[2];
    const float zz = A[3] * (1.f / 3.f);
    Tn[0] = 0.5f * (A[6] - zz); Tn[1] = 0.5f * (-A[6] - zz); Tn[2] = zz;
    Tn[3] = 0.5f * A[7]; Tn[4] = A[4]; Tn[5] = A[5];
    Sn[0] = Tn[0] * Tn[0] + Tn[3] * Tn[3] + Tn[4] * Tn[4];
    Sn[1] = Tn[3] * Tn[3] + Tn[1] * Tn[1] + Tn[5] * Tn[5];
    Sn[2] = Tn[4] * Tn[4] + Tn[5] * Tn[5] + Tn[2] * Tn[2];
    Sn[3] = Tn[0] * Tn[3] + Tn[3] * Tn[1] + Tn[4] * Tn[5];
    Sn[4] = Tn[0] * Tn[4] + Tn[3] * Tn[5] + Tn[4] * Tn[2];
    Sn[5] = Tn[3] * Tn[4] + Tn[1] * Tn[5] + Tn[5] * Tn[2];
}

template <int T, bool ZBL>
__global__ void __launch_bounds__(ANG_BLOCK)
k_desc_angular(int64_t N, const float4* __restrict__ xyzt, const float4* __restrict__ lvA, int capLA, const int* __restrict__ nlvA,
               const float* __restrict__ cA, float rcinv, float* __restrict__ D, float* __restrict__ Aout,
               ZblParams zbl, double* __restrict__ sums, int hb /* 4-/5-body terms on: rows 25..34 of D */)
{
    // g_n = sum_k c_nk f_k = 1/2 fc [ (2 c_n0 + sum_{k>=1} c_nk) + sum_{k>=1} c_nk T_k ]: row (ti, tj, n) of the table holds the
    // bracket's constant in slot 0 and c_n1..c_n8 behind it, so g_n is a dot product with (1, T_1..T_8) in packed FMAs and the
    // basis functions f_k themselves are never formed.
    __shared__ __align__(16) float sh_c[T * T * NR * KP];
    __shared__ float4 sh_ring[ANG_DEPTH][ANG_BLOCK];
    for (int i = threadIdx.x; i < T * T * NR; i += blockDim.x) {
        const float* c = cA + i * KP;
        float c0 = 2.f * c[0];
#pragma unroll
        for (int k = 1; k < NB; ++k) { c0 += c[k]; sh_c[i * KP + k] = c[k]; }
        sh_c[i * KP] = c0;
        sh_c[i * KP + 9] = 0.f; sh_c[i * KP + 10] = 0.f; sh_c[i * KP + 11] = 0.f;
    }
    __syncthreads();
    const int64_t p0 = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool live = p0 < N;                                // threads beyond N stay for the warp sum of the ZBL energy
    const int64_t p = live ? p0 : N - 1;
    const int ti = __float_as_int(xyzt[p].w);
    float ezbl = 0.f;                                        // 1/2 sum_j U_ZBL(r_ij) of this atom (qnep_set_zbl)
    // accumulators as register pairs: the 120 updates A_nlm += g_n b_lm of a neighbour are 60 packed FMAs (FFMA2:
    // two FP32 FMAs per issued instruction; this kernel is bound by issue slots, not by latency)
    float2 A2[NR][NLM / 2];
#pragma unroll
    for (int a = 0; a < NR; ++a)
#pragma unroll
        for (int m = 0; m < NLM / 2; ++m) A2[a][m] = make_float2(0.f, 0.f);
    const int n = live ? nlvA[p] : 0;
    const float4* rows = lvA + qnep_tiled_base(p, capLA);
    const int tid = threadIdx.x;
#pragma unroll
    for (int k = 0; k < ANG_DEPTH; ++k) {
        if (k < n) cp_async16_cg(&sh_ring[k][tid], rows + (int64_t)k * QNEP_TILE);
        cp_async_commit();
    }
    for (int s = 0; s < n; ++s) {
        cp_async_wait<ANG_DEPTH - 1>();
        const float4 pr = sh_ring[s & (ANG_DEPTH - 1)][tid];
        if (s + ANG_DEPTH < n) cp_async16_cg(&sh_ring[s & (ANG_DEPTH - 1)][tid], rows + (int64_t)(s + ANG_DEPTH) * QNEP_TILE);
        cp_async_commit();
        const float r2 = pr.x * pr.x + pr.y * pr.y + pr.z * pr.z;
        const float rinv = fast_rsqrt(r2), r = r2 * rinv;
        if (ZBL && r2 < zbl.r2sq) {
            float u, du;
            qnep_zbl_eval(zbl, ti, (int)((unsigned)__float_as_int(pr.w) >> QNEP_NL_SHIFT), r, rinv, u, du);
            ezbl = fmaf(0.5f, u, ezbl);
        }
        const float tt = r * rcinv;
        const float hfc = 0.25f + 0.25f * __cosf(3.14159265358979f * tt);
        const float tm1 = tt - 1.f;
        const float xx = 2.f * tm1 * tm1 - 1.f, xx2 = xx + xx;
        float Tk[NB];                                    // T_1 .. T_8 in Tk[1..8]
        Tk[0] = 1.f; Tk[1] = xx;
#pragma unroll
        for (int k = 2; k < NB; ++k) Tk[k] = fmaf(xx2, Tk[k - 1], -Tk[k - 2]);
        const int tj = (unsigned)__float_as_int(pr.w) >> QNEP_NL_SHIFT;
        const float4* c4 = reinterpret_cast<const float4*>(sh_c + (ti * T + tj) * NR * KP);
        float2 g2[NR];
#pragma unroll
        for (int a = 0; a < NR; ++a) {
            const float4 ca = c4[a * 3], cb = c4[a * 3 + 1], cc = c4[a * 3 + 2];      // (c0', c1, c2, c3) (c4..c7) (c8, 0, 0, 0)
            float2 v = __fmul2_rn(make_float2(ca.x, ca.y), make_float2(Tk[0], Tk[1]));     // aligned pairs of the float4 rows
            v = __ffma2_rn(make_float2(ca.z, ca.w), make_float2(Tk[2], Tk[3]), v);
            v = __ffma2_rn(make_float2(cb.x, cb.y), make_float2(Tk[4], Tk[5]), v);
            v = __ffma2_rn(make_float2(cb.z, cb.w), make_float2(Tk[6], Tk[7]), v);
            const float g = hfc * fmaf(cc.x, Tk[8], v.x + v.y);
            g2[a] = make_float2(g, g);
        }
        float b[NLM];
        harmonics(pr.x * rinv, pr.y * rinv, pr.z * rinv, b);
#pragma unroll
        for (int a = 0; a < NR; ++a)
#pragma unroll
            for (int m = 0; m < NLM / 2; ++m) A2[a][m] = __ffma2_rn(g2[a], make_float2(b[2 * m], b[2 * m + 1]), A2[a][m]);
    }
    if (ZBL) {
        double e = (double)ezbl;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
        if ((tid & 31) == 0 && e != 0.0) atomicAdd(&sums[SUM_COUNT + (blockIdx.x % QNEP_WSTRIPES) * QNEP_WSTRIDE + 9], e);
    }
    if (!live) return;
#pragma unroll
    for (int a = 0; a < NR; ++a) {
        float d[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int lm = 0; lm < NLM; ++lm) {
            const float Av = (lm & 1) ? A2[a][lm >> 1].y : A2[a][lm >> 1].x;
            d[l_of_lm(lm)] = fmaf(c_Clm[lm] * Av, Av, d[l_of_lm(lm)]);
            Aout[(int64_t)(a * NLM + lm) * N + p] = Av;
        }
#pragma unroll
        for (int l = 0; l < 4; ++l) D[(int64_t)(NR + a * 4 + l) * N + p] = d[l];
        if (hb) {
            float A8[8], Tn[6], Sn[6], w2;
#pragma unroll
            for (int lm = 0; lm < 8; ++lm) A8[lm] = (lm & 1) ? A2[a][lm >> 1].y : A2[a][lm >> 1].x;
            hb_moments(A8, Tn, Sn, w2);
            // 4-body: tr(T^3) = sum_ab S_ab T_ab;  5-body: (w.w)^2
            D[(int64_t)(ND + a) * N + p] = Sn[0] * Tn[0] + Sn[1] * Tn[1] + Sn[2] * Tn[2] + 2.f * (Sn[3] * Tn[3] + Sn[4] * Tn[4] + Sn[5] * Tn[5]);
            D[(int64_t)(ND + NR + a) * N + p] = w2 * w2;
        }
    }
}

// ------------------------------------------------------------------------------------------
// a4 (+a10 in two halves): NN forward, dU/dD and dq/dD.  Weights per type in shared memory:
//   w0s[H][28] (= w0 * scaler, rows padded to 28), b0[H], w1U[H], w1q[H]
// ------------------------------------------------------------------------------------------
constexpr int W0P = 28;

__device__ __forceinline__ float tanh_f32(float z)
{
    // tanh z = 1 - 2 / (exp(2z) + 1) on the MUFU pipe (EX2, RCP); exact limits at +-inf.  Where the exponent is
    // large the result is insensitive to it, so the fp32 rounding of 2 z log2(e) costs < 1e-7 absolute.
    float e, r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(z * 2.885390081777927f));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(e + 1.f));
    return fmaf(-2.f, r, 1.f);
}

// Persistent blocks: the weights of all species are staged in shared memory once per block, then the block walks
// chunks of 2 x 128 atoms.  A thread owns TWO atoms (p and p + 128 of the chunk) and keeps their descriptors and both
// derivative vectors as register pairs (atom A, atom B): a weight read from shared memory serves both atoms, and every
// update is one packed FMA (FFMA2) with the weight or the per-atom factor as the scalar operand -- half the issue
// slots per atom of the scalar form, which was bound by issue slots (77 % busy, FMA pipe 63 %).  The two atoms of a
// thread are of one species except where a chunk straddles a species boundary of the sorted order; there the hidden
// layer is evaluated once per species with the other atom masked out.
constexpr int NN_BLOCK = 128;
#ifndef QNEP_NN_UNROLL
#define QNEP_NN_UNROLL 2
#endif
constexpr int NN_UNROLL = QNEP_NN_UNROLL;

#ifndef QNEP_NN_MINB
#define QNEP_NN_MINB 2
#endif
__global__ void __launch_bounds__(NN_BLOCK, QNEP_NN_MINB)
k_nn(int64_t N, int T, int H, int nn_stride, const float* __restrict__ nnw, float b1U, float b1q,
     const float4* __restrict__ xyzt, const float* __restrict__ D, float* __restrict__ Ui, float* __restrict__ qraw,
     float* __restrict__ FpU, float* __restrict__ FpQ, double* __restrict__ sums)
{
    extern __shared__ __align__(16) float sh_w[];
    __shared__ double sh_red[32];
    {
        const float4* src = reinterpret_cast<const float4*>(nnw);
        float4* dst = reinterpret_cast<float4*>(sh_w);
        for (int i = threadIdx.x; i < T * nn_stride / 4; i += blockDim.x) dst[i] = src[i];
    }
    __syncthreads();
    double accU = 0.0, accQ = 0.0;
    const int64_t nchunk = (N + 2 * NN_BLOCK - 1) / (2 * NN_BLOCK);
    for (int64_t ch = blockIdx.x; ch < nchunk; ch += gridDim.x) {
        const int64_t pA = ch * (2 * NN_BLOCK) + threadIdx.x, pB = pA + NN_BLOCK;
        const bool okA = pA < N, okB = pB < N;
        const int64_t qA = okA ? pA : N - 1, qB = okB ? pB : N - 1;
        const int tA = __float_as_int(xyzt[qA].w), tB = __float_as_int(xyzt[qB].w);
        float2 x[ND], dU[ND], dQ[ND];
#pragma unroll
        for (int v = 0; v < ND; ++v) {
            x[v] = make_float2(D[(int64_t)v * N + qA], D[(int64_t)v * N + qB]);
            dU[v] = make_float2(0.f, 0.f);
            dQ[v] = make_float2(0.f, 0.f);
        }
        float2 U = make_float2(0.f, 0.f), q = make_float2(0.f, 0.f);
        const int npass = tA == tB ? 1 : 2;
        for (int pass = 0; pass < npass; ++pass) {
            const float* w = sh_w + (pass == 0 ? tA : tB) * nn_stride;
            const float* b0 = w + H * W0P;
            const float* w1U = b0 + H;
            const float* w1q = w1U + H;
            // which of the two atoms this pass serves (both when the species agree)
            const float2 on = npass == 1 ? make_float2(1.f, 1.f) : (pass == 0 ? make_float2(1.f, 0.f) : make_float2(0.f, 1.f));
#pragma unroll NN_UNROLL
            for (int mu = 0; mu < H; ++mu) {
                const float4* row = reinterpret_cast<const float4*>(w + mu * W0P);
                float wr[W0P];
#pragma unroll
                for (int v4 = 0; v4 < W0P / 4; ++v4) {
                    const float4 t = row[v4];
                    wr[4 * v4] = t.x; wr[4 * v4 + 1] = t.y; wr[4 * v4 + 2] = t.z; wr[4 * v4 + 3] = t.w;
                }
                const float nb0 = -b0[mu];
                float2 zc[4] = {make_float2(nb0, nb0), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};   // four chains
#pragma unroll
                for (int v = 0; v < ND; ++v) zc[v & 3] = __ffma2_rn(make_float2(wr[v], wr[v]), x[v], zc[v & 3]);
                const float2 zs = __fadd2_rn(__fadd2_rn(zc[0], zc[1]), __fadd2_rn(zc[2], zc[3]));
                const float2 h2 = make_float2(tanh_f32(zs.x), tanh_f32(zs.y));
                const float a = w1U[mu], b = w1q[mu];
                const float2 a2 = make_float2(a * on.x, a * on.y), b2 = make_float2(b * on.x, b * on.y);
                U = __ffma2_rn(a2, h2, U);
                q = __ffma2_rn(b2, h2, q);
                const float2 dh = make_float2(fmaf(-h2.x, h2.x, 1.f), fmaf(-h2.y, h2.y, 1.f));
                const float2 au = __fmul2_rn(a2, dh), bq = __fmul2_rn(b2, dh);
#pragma unroll
                for (int v = 0; v < ND; ++v) {
                    const float2 wv = make_float2(wr[v], wr[v]);
                    dU[v] = __ffma2_rn(au, wv, dU[v]);
                    dQ[v] = __ffma2_rn(bq, wv, dQ[v]);
                }
            }
        }
        U.x -= b1U; U.y -= b1U;
        q.x -= b1q; q.y -= b1q;
        if (okA) {
            Ui[pA] = U.x; qraw[pA] = q.x;
#pragma unroll
            for (int v = 0; v < ND; ++v) { FpU[(int64_t)v * N + pA] = dU[v].x; FpQ[(int64_t)v * N + pA] = dQ[v].x; }
            accU += (double)U.x; accQ += (double)q.x;
        }
        if (okB) {
            Ui[pB] = U.y; qraw[pB] = q.y;
#pragma unroll
            for (int v = 0; v < ND; ++v) { FpU[(int64_t)v * N + pB] = dU[v].y; FpQ[(int64_t)v * N + pB] = dQ[v].y; }
            accU += (double)U.y; accQ += (double)q.y;
        }
    }
    const double su = block_sum(accU, sh_red);
    const double sq = block_sum(accQ, sh_red);
    if (threadIdx.x == 0) { atomicAdd(&sums[SUM_E_NEP], su); atomicAdd(&sums[SUM_Q], sq); }
}

// ------------------------------------------------------------------------------------------
// a4 on the tensor cores (the one stage where the north_star allows them): the batched contraction
//   Z[atoms x H] = X[atoms x 25] W0^T,   dU/dD[atoms x 25] = (w1U (1 - h^2))[atoms x H] W0,   dq/dD likewise
// as warp-level mma.sync m16n8k8 TF32 with the 3xTF32 split (x = hi + lo, three products per term: the error of a product is
// ~2^-21 relative, the level of the FP32 form, so the 1e-5 eV/atom energy tolerance holds -- measured in the parity tests).
// A warp owns 32 atoms (two m16 tiles).  Per block of eight neurons: 24 mma give z, the activation and the two output
// sums run on the accumulator fragment, and that fragment IS the A operand of the backward products for these eight
// neurons (accumulator element (row, col 2t / 2t+1) = A element (row, k = t / t+4) once the neurons of the block are
// taken in the order 0 2 4 6 1 3 5 7, which the B operand read from shared memory follows): no data movement.
// Weights are split into hi / lo once per block, rows padded to 36 floats (conflict-free fragment reads).
// ------------------------------------------------------------------------------------------
constexpr int NNM_LD = 36;            // padded row of the split weight tables
constexpr int NNM_K = 32;             // descriptors padded to four k-steps of eight

__device__ __forceinline__ unsigned tf32_hi(float x) { unsigned r; asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x)); return r; }
__device__ __forceinline__ void tf32_split(float x, unsigned& hi, unsigned& lo)
{
    hi = tf32_hi(x);
    lo = tf32_hi(x - __uint_as_float(hi));
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const unsigned (&a)[4], unsigned b0, unsigned b1)
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__global__ void __launch_bounds__(128, 2)      // 242 registers; 1, 3 and 4 blocks per SM are slower (0.44 / 0.39 / 0.45 ms)
k_nn_mma(int64_t N, int T, int H, int HP /* H rounded up to 8 */, int nn_stride, const float* __restrict__ nnw, float b1U, float b1q,
         const float4* __restrict__ xyzt, const float* __restrict__ D, float* __restrict__ Ui, float* __restrict__ qraw,
         float* __restrict__ FpU, float* __restrict__ FpQ, double* __restrict__ sums)
{
    extern __shared__ __align__(16) float sh_nn[];
    // per type: Wh[HP][NNM_LD], Wl[HP][NNM_LD], b0[HP], w1U[HP], w1q[HP]
    const int tstride = 2 * HP * NNM_LD + 3 * HP;
    __shared__ double sh_red[32];
    for (int i = threadIdx.x; i < T * tstride; i += blockDim.x) sh_nn[i] = 0.f;
    __syncthreads();
    for (int t = 0; t < T; ++t) {
        const float* w = nnw + (size_t)t * nn_stride;            // w0s[H][W0P], b0[H], w1U[H], w1q[H]
        float* dst = sh_nn + t * tstride;
        for (int i = threadIdx.x; i < H * ND; i += blockDim.x) {
            const int mu = i / ND, v = i - mu * ND;
            unsigned hi, lo;
            tf32_split(w[mu * W0P + v], hi, lo);
            dst[mu * NNM_LD + v] = __uint_as_float(hi);
            dst[HP * NNM_LD + mu * NNM_LD + v] = __uint_as_float(lo);
        }
        for (int i = threadIdx.x; i < 3 * H; i += blockDim.x) dst[2 * HP * NNM_LD + (i / H) * HP + (i % H)] = w[H * W0P + i];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int g = lane >> 2, t4 = lane & 3;
    double accU = 0.0, accQ = 0.0;
    const int64_t nwtile = (N + 31) / 32;
    for (int64_t wt = (int64_t)blockIdx.x * 4 + wib; wt < nwtile; wt += (int64_t)gridDim.x * 4) {
        const int64_t a0 = wt * 32;
        // rows of this lane: r = 0..3 -> atom a0 + g + 8 r  (m-tile r / 2, fragment row g + 8 (r & 1))
        int64_t atom[4];
        int typ[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            atom[r] = min(a0 + g + 8 * r, N - 1);
            typ[r] = __float_as_int(xyzt[atom[r]].w);
        }
        // X fragments, split: xa[m][ks][4]
        unsigned xh[2][4][4], xl[2][4][4];
#pragma unroll
        for (int m = 0; m < 2; ++m)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int v = 8 * ks + t4 + 4 * (e >> 1);
                    const float x = v < ND ? D[(int64_t)v * N + atom[2 * m + (e & 1)]] : 0.f;
                    tf32_split(x, xh[m][ks][e], xl[m][ks][e]);
                }
        // which species does the warp hold?  (one, except at a species boundary of the sorted order)
        unsigned present = 0;
#pragma unroll
        for (int r = 0; r < 4; ++r) present |= 1u << typ[r];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) present |= __shfl_xor_sync(0xffffffffu, present, o);
        for (int ty = 0; ty < T; ++ty) {
            if (!((present >> ty) & 1u)) continue;
            const float* Wh = sh_nn + ty * tstride;
            const float* Wl = Wh + HP * NNM_LD;
            const float* b0 = Wl + HP * NNM_LD;
            const float* w1U = b0 + HP;
            const float* w1q = w1U + HP;
            float dU[2][4][4], dQ[2][4][4], U[4] = {0.f, 0.f, 0.f, 0.f}, q[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int m = 0; m < 2; ++m)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                    for (int e = 0; e < 4; ++e) { dU[m][nt][e] = 0.f; dQ[m][nt][e] = 0.f; }
            for (int j = 0; j < HP / 8; ++j) {
                // forward: z[m] = X W0^T for neurons 8 j .. 8 j + 7 (B element (k, n) = w0[8 j + n][k])
                // (three accumulators per tile: the mma latency is ~30 cycles and only two warps share a scheduler)
                float z[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
                float zb[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}}, zc[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                    const int o0 = (8 * j + g) * NNM_LD + 8 * ks + t4;
                    const unsigned bh0 = __float_as_uint(Wh[o0]), bh1 = __float_as_uint(Wh[o0 + 4]);
                    const unsigned bl0 = __float_as_uint(Wl[o0]), bl1 = __float_as_uint(Wl[o0 + 4]);
#pragma unroll
                    for (int m = 0; m < 2; ++m) {
                        mma_tf32(zb[m], xl[m][ks], bh0, bh1);
                        mma_tf32(zc[m], xh[m][ks], bl0, bl1);
                        mma_tf32(z[m], xh[m][ks], bh0, bh1);
                    }
                }
#pragma unroll
                for (int m = 0; m < 2; ++m)
#pragma unroll
                    for (int e = 0; e < 4; ++e) z[m][e] += zb[m][e] + zc[m][e];
                // activation on the accumulator fragment: element e of tile m = (row g + 8 (e >> 1), neuron 8 j + 2 t4 + (e & 1))
                unsigned auh[2][4], aul[2][4], bqh[2][4], bql[2][4];
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int mu = 8 * j + 2 * t4 + c;
                    const float bb = b0[mu], aU = w1U[mu], aQ = w1q[mu];
#pragma unroll
                    for (int m = 0; m < 2; ++m)
#pragma unroll
                        for (int rr = 0; rr < 2; ++rr) {
                            const float hmu = tanh_f32(z[m][2 * rr + c] - bb);
                            U[2 * m + rr] = fmaf(aU, hmu, U[2 * m + rr]);
                            q[2 * m + rr] = fmaf(aQ, hmu, q[2 * m + rr]);
                            const float dh = fmaf(-hmu, hmu, 1.f);
                            // A fragment of the backward product: (row g + 8 rr, k = t4 + 4 c)  ->  register rr + 2 c
                            tf32_split(aU * dh, auh[m][rr + 2 * c], aul[m][rr + 2 * c]);
                            tf32_split(aQ * dh, bqh[m][rr + 2 * c], bql[m][rr + 2 * c]);
                        }
                }
                // backward: dU += AU W0, dQ += BQ W0 over these eight neurons (B element (k, n) = w0[8 j + pi(k)][8 nt + n],
                // pi(k) = 2 k for k < 4, 2 (k - 4) + 1 else: the order the accumulator fragment holds them in)
#pragma unroll
                for (int nt = 0; nt < 4; ++nt) {
                    const int o0 = (8 * j + 2 * t4) * NNM_LD + 8 * nt + g;
                    const unsigned bh0 = __float_as_uint(Wh[o0]), bh1 = __float_as_uint(Wh[o0 + NNM_LD]);
                    const unsigned bl0 = __float_as_uint(Wl[o0]), bl1 = __float_as_uint(Wl[o0 + NNM_LD]);
#pragma unroll
                    for (int m = 0; m < 2; ++m) {
                        mma_tf32(dU[m][nt], aul[m], bh0, bh1);
                        mma_tf32(dU[m][nt], auh[m], bl0, bl1);
                        mma_tf32(dU[m][nt], auh[m], bh0, bh1);
                        mma_tf32(dQ[m][nt], bql[m], bh0, bh1);
                        mma_tf32(dQ[m][nt], bqh[m], bl0, bl1);
                        mma_tf32(dQ[m][nt], bqh[m], bh0, bh1);
                    }
                }
            }
            // the two output sums: a lane holds two of the eight neurons of every block, the quad holds all
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                U[r] += __shfl_xor_sync(0xffffffffu, U[r], 1); U[r] += __shfl_xor_sync(0xffffffffu, U[r], 2);
                q[r] += __shfl_xor_sync(0xffffffffu, q[r], 1); q[r] += __shfl_xor_sync(0xffffffffu, q[r], 2);
            }
            // outputs of the rows of this species: accumulator element (row r, descriptor 8 nt + 2 t4 + c)
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int64_t p = a0 + g + 8 * r;
                if (p < N && typ[r] == ty) {
                    const float Uv = U[r] - b1U, qv = q[r] - b1q;
                    if (t4 == 0) { Ui[p] = Uv; qraw[p] = qv; accU += (double)Uv; accQ += (double)qv; }
#pragma unroll
                    for (int nt = 0; nt < 4; ++nt)
#pragma unroll
                        for (int c = 0; c < 2; ++c) {
                            const int v = 8 * nt + 2 * t4 + c;
                            if (v < ND) {
                                FpU[(int64_t)v * N + p] = dU[r >> 1][nt][2 * (r & 1) + c];
                                FpQ[(int64_t)v * N + p] = dQ[r >> 1][nt][2 * (r & 1) + c];
                            }
                        }
                }
            }
        }
    }
    const double su = block_sum(accU, sh_red);
    const double sq = block_sum(accQ, sh_red);
    if (threadIdx.x == 0) { atomicAdd(&sums[SUM_E_NEP], su); atomicAdd(&sums[SUM_Q], sq); }
}

// ------------------------------------------------------------------------------------------
// a4 on the 5th-generation tensor cores: tcgen05.mma kind::tf32 with accumulators AND the A operands in tensor memory.
// A block of 128 threads owns 128 atoms of ONE species (tiles are cut per species range of the sorted order); thread r is
// row r of every matrix, i.e. TMEM lane r:
//   1. x (25 descriptors, padded to 32) is split into TF32 hi / lo and written to TMEM columns with tcgen05.st;
//   2. one thread issues Z = X W0^T as 3 x 4 MMAs (M = 128, N = HP neurons, K = 8; A from TMEM, B = the split weights in
//      shared memory, K-major canonical layout without swizzle), commits to an mbarrier;
//   3. per chunk of 16 neurons every thread reads its 16 z values (tcgen05.ld), applies the activation, adds to its U and q,
//      splits a (1 - h^2) for both outputs into hi / lo and stores them to TMEM as the A operand of the backward products
//      dU/dD += AU W0, dq/dD += BQ W0 (N = 32 descriptors, K = 16), issued by one thread;
//   4. dU/dD, dq/dD come back with tcgen05.ld, one row per thread, and go to FpU / FpQ with coalesced stores.
// 3xTF32 keeps FP32-level accuracy (see k_nn_mma).  TMEM columns: Z [0, HP), operand staging [128, 192), dU [192, 224),
// dQ [224, 256): 256 columns per block, two blocks per SM.
// ------------------------------------------------------------------------------------------
constexpr int UM_COL_A = 128, UM_COL_DU = 192, UM_COL_DQ = 224, UM_COLS = 256;

__device__ __forceinline__ uint64_t umma_smem_desc(unsigned smem_addr, unsigned lbo_bytes, unsigned sbo_bytes)
{
    // start address, leading-dimension byte offset, stride byte offset (each >> 4), version 1 (Blackwell), no swizzle
    return (uint64_t)((smem_addr >> 4) & 0x3fff) | ((uint64_t)((lbo_bytes >> 4) & 0x3fff) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3fff) << 32) | (1ull << 46);
}
__device__ __forceinline__ void umma_tf32_ts(unsigned tmem_d, unsigned tmem_a, uint64_t desc_b, unsigned idesc, unsigned accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}\n"
                 ::"r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void tmem_st16(unsigned taddr, const unsigned (&v)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]),
                   "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_ld16(unsigned taddr, float (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7]), "=f"(v[8]),
                   "=f"(v[9]), "=f"(v[10]), "=f"(v[11]), "=f"(v[12]), "=f"(v[13]), "=f"(v[14]), "=f"(v[15]) : "r"(taddr) : "memory");
}
// split for operands formed on the fly: hi = x with the 13 low mantissa bits cleared (what the tensor core reads of a TF32
// container anyway), lo = x - hi exactly; the hardware truncates lo to TF32 itself (error 2^-20 of x).  Two instructions.
__device__ __forceinline__ void tf32_split_trunc(float x, unsigned& hi, unsigned& lo)
{
    hi = __float_as_uint(x) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}
// wait for the mbarrier phase; a bounded spin so that a faulting MMA cannot hang the device (flag -> QNEP_ERR_CUDA)
__device__ __forceinline__ bool mbar_wait(unsigned bar, unsigned parity)
{
    for (int spin = 0; spin < (1 << 20); ++spin) {
        unsigned ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}\n"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return true;
    }
    return false;
}

__global__ void __launch_bounds__(128, 2)
k_nn_umma(int64_t N, int T, int H, int HP /* H rounded up to 16 */, int nn_stride, const float* __restrict__ nnw, float b1U, float b1q,
          const int* __restrict__ start /* [T * ncells + 1] first sorted index of every (species, cell) bucket */, int ncells,
          const float* __restrict__ D, float* __restrict__ Ui, float* __restrict__ qraw,
          float* __restrict__ FpU, float* __restrict__ FpQ, double* __restrict__ sums, int* __restrict__ flags)
{
    extern __shared__ __align__(128) unsigned char sh_um[];
    // forward B (rows = neurons, K = 32 descriptors): [8 chunks][HP][4] hi, then lo; backward B (rows = 32 descriptors, K = HP
    // neurons): [HP / 4 chunks][32][4] hi, then lo; then b0, w1U, w1q [HP]
    // (backward: both outputs share the factor 1 - h^2, so the A operand is dh alone and the output weights are folded into two
    //  B tables, WU = w1U_mu w0[mu][v] and WQ = w1q_mu w0[mu][v]: one split and one staging store per neuron instead of two)
    float* Wf_h = reinterpret_cast<float*>(sh_um);
    float* Wf_l = Wf_h + 32 * HP;
    // backward B: ONE table of 64 rows (rows 0..31: WU of descriptor v, rows 32..63: WQ), [HP / 4 chunks][64][4], so that
    // dU/dD and dq/dD are the 64 columns of one accumulator and one MMA (N = 64) serves both
    float* WB_h = Wf_l + 32 * HP;
    float* WB_l = WB_h + 64 * HP;
    float4* nc = reinterpret_cast<float4*>(WB_l + 64 * HP);      // per neuron (b0, w1U, w1q, 0)
    __shared__ __align__(8) unsigned long long sh_bar[3];     // [0] forward products, [1], [2] backward products of even / odd chunks
    __shared__ unsigned sh_tmem;
    __shared__ double sh_red[32];
    __shared__ int sh_ts[QNEP_MAX_TYPES + 1];
    const int tid = threadIdx.x, warp = tid >> 5;
    const unsigned bar = (unsigned)__cvta_generic_to_shared(&sh_bar[0]);     // a waiter may lag ONE phase behind a barrier: one barrier per buffer
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(&sh_tmem)), "n"(UM_COLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tid == 0) {
        for (int i = 0; i < 3; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar + 8 * i));
        asm volatile("fence.mbarrier_init.release.cluster;");
        for (int t = 0; t <= T; ++t) sh_ts[t] = t < T ? start[t * ncells] : (int)N;
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const unsigned tbase = sh_tmem + ((unsigned)(32 * warp) << 16);       // this warp's lanes
    const unsigned tbase0 = sh_tmem;
    const unsigned idesc_f = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(HP >> 3) << 17) | (8u << 24);    // F32 accum, TF32 x TF32, N = HP, M = 128
    const unsigned idesc_b = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(64 >> 3) << 17) | (8u << 24);    // N = 64
    const unsigned wf_h = (unsigned)__cvta_generic_to_shared(Wf_h), wf_l = (unsigned)__cvta_generic_to_shared(Wf_l);
    const unsigned wb_h = (unsigned)__cvta_generic_to_shared(WB_h), wb_l = (unsigned)__cvta_generic_to_shared(WB_l);
    // tiles: species t has ceil(n_t / 128) tiles
    int ntile_t[QNEP_MAX_TYPES], ntiles = 0;
    for (int t = 0; t < T; ++t) { ntile_t[t] = (sh_ts[t + 1] - sh_ts[t] + 127) / 128; ntiles += ntile_t[t]; }
    unsigned phase = 0, phc[2] = {0, 0};
    int loaded_type = -1;
    bool ok = true;
    double accU = 0.0, accQ = 0.0;
    // descriptors of a tile are requested one tile ahead (they were 8 % of the stalls when loaded at the point of use)
    float xn[ND];
    auto tile_row = [&](int tile, int& ty) -> int64_t {
        int rel = tile;
        ty = 0;
        while (rel >= ntile_t[ty]) { rel -= ntile_t[ty]; ++ty; }
        return sh_ts[ty] + (int64_t)rel * 128;
    };
    auto request = [&](int tile) {
        if (tile >= ntiles) return;
        int ty;
        const int64_t pp = tile_row(tile, ty) + tid;
        const bool lv = pp < sh_ts[ty + 1];
#pragma unroll
        for (int v = 0; v < ND; ++v) xn[v] = lv ? D[(int64_t)v * N + pp] : 0.f;
    };
    request(blockIdx.x);
    for (int tile = blockIdx.x; tile < ntiles && ok; tile += gridDim.x) {
        int ty;
        const int64_t row0 = tile_row(tile, ty);
        const int64_t p = row0 + tid;
        const bool live = p < sh_ts[ty + 1];
        if (ty != loaded_type) {
            // (the previous tile's MMAs have completed: every tile ends with a wait on the barrier)
            const float* w = nnw + (size_t)ty * nn_stride;
            for (int i = tid; i < 32 * HP; i += blockDim.x) {
                const int mu = i / 32, v = i - mu * 32;
                const float x = (mu < H && v < ND) ? w[mu * W0P + v] : 0.f;
                const float aU = mu < H ? w[H * W0P + H + mu] : 0.f, aQ = mu < H ? w[H * W0P + 2 * H + mu] : 0.f;
                unsigned hi, lo;
                tf32_split(x, hi, lo);
                const int of = (v >> 2) * HP * 4 + mu * 4 + (v & 3);         // forward B: row mu, k = v
                const int ob = (mu >> 2) * 64 * 4 + v * 4 + (mu & 3);        // backward B: row v (WU) / 32 + v (WQ), k = mu
                Wf_h[of] = __uint_as_float(hi); Wf_l[of] = __uint_as_float(lo);
                tf32_split(aU * x, hi, lo);
                WB_h[ob] = __uint_as_float(hi); WB_l[ob] = __uint_as_float(lo);
                tf32_split(aQ * x, hi, lo);
                WB_h[ob + 32 * 4] = __uint_as_float(hi); WB_l[ob + 32 * 4] = __uint_as_float(lo);
            }
            for (int i = tid; i < HP; i += blockDim.x)
                nc[i] = i < H ? make_float4(w[H * W0P + i], w[H * W0P + H + i], w[H * W0P + 2 * H + i], 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
            loaded_type = ty;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the tensor core
        }
        // 1. X hi / lo to TMEM columns UM_COL_A .. +32 and +32 .. +64
        {
            unsigned xh[32], xl[32];
#pragma unroll
            for (int v = 0; v < 32; ++v) tf32_split_trunc(v < ND ? xn[v] : 0.f, xh[v], xl[v]);
            request(tile + gridDim.x);
            tmem_st16(tbase + UM_COL_A, reinterpret_cast<const unsigned (&)[16]>(xh[0]));
            tmem_st16(tbase + UM_COL_A + 16, reinterpret_cast<const unsigned (&)[16]>(xh[16]));
            tmem_st16(tbase + UM_COL_A + 32, reinterpret_cast<const unsigned (&)[16]>(xl[0]));
            tmem_st16(tbase + UM_COL_A + 48, reinterpret_cast<const unsigned (&)[16]>(xl[16]));
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        // 2. forward products
        if (tid == 0) {
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                const uint64_t dh = umma_smem_desc(wf_h + 2 * ks * HP * 16, HP * 16, 128), dl = umma_smem_desc(wf_l + 2 * ks * HP * 16, HP * 16, 128);
                umma_tf32_ts(tbase0, tbase0 + UM_COL_A + 32 + 8 * ks, dh, idesc_f, ks > 0);      // x_lo w_hi
                umma_tf32_ts(tbase0, tbase0 + UM_COL_A + 8 * ks, dl, idesc_f, 1);                // x_hi w_lo
                umma_tf32_ts(tbase0, tbase0 + UM_COL_A + 8 * ks, dh, idesc_f, 1);                // x_hi w_hi
            }
            asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
        }
        ok = mbar_wait(bar, phase);
        phase ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // 3. activation per chunk of 16 neurons, backward products
        float U = 0.f, q = 0.f;
        // (after a timed-out wait the chunk loop still runs to its end: every warp keeps its named-barrier arrivals, so a
        // thread that saw the time-out and one that did not cannot strand each other; the later waits return at once)
        for (int c = 0; c < HP / 16; ++c) {
            float z[16];
            tmem_ld16(tbase + 16 * c, z);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            unsigned dhh[16], dhl[16];
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const int mu = 16 * c + k;
                const float4 cn = nc[mu];
                const float hmu = tanh_f32(z[k] - cn.x);
                U = fmaf(cn.y, hmu, U);
                q = fmaf(cn.z, hmu, q);
                tf32_split_trunc(fmaf(-hmu, hmu, 1.f), dhh[k], dhl[k]);
            }
            // two staging buffers of 32 columns (chunk parity): buffer c & 1 is free once the products of chunk c - 2 have
            // completed, so the activation runs up to two chunks ahead of the tensor core
            if (c > 1) {
                ok = ok && mbar_wait(bar + 8 + 8 * (c & 1), phc[c & 1]);
                phc[c & 1] ^= 1;
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            }
            const unsigned stg = UM_COL_A + 32 * (c & 1);
            tmem_st16(tbase + stg, dhh);
            tmem_st16(tbase + stg + 16, dhl);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            // the issuing warp waits for the staging stores of all four warps; the other warps only announce theirs and go on
            // to the activation of the next chunk
            // (two named barriers by chunk parity: the other warps may be one chunk ahead of the issuing warp)
            if (warp == 0) asm volatile("bar.sync %0, 128;" ::"r"(1 + (c & 1)) : "memory");
            else asm volatile("bar.arrive %0, 128;" ::"r"(1 + (c & 1)) : "memory");
            if (tid == 0) {
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll
                for (int k2 = 0; k2 < 2; ++k2) {
                    const int kk = 2 * c + k2;                                                   // k-step of eight neurons
                    const uint64_t bh = umma_smem_desc(wb_h + 2 * kk * 1024, 1024, 128), bl = umma_smem_desc(wb_l + 2 * kk * 1024, 1024, 128);
                    const unsigned acc = (c > 0 || k2 > 0) ? 1u : 0u;
                    const unsigned a_hi = tbase0 + stg + 8 * k2, a_lo = tbase0 + stg + 16 + 8 * k2;
                    umma_tf32_ts(tbase0 + UM_COL_DU, a_lo, bh, idesc_b, acc);      // dh_lo W_hi   (columns: dU/dD, then dq/dD)
                    umma_tf32_ts(tbase0 + UM_COL_DU, a_hi, bl, idesc_b, 1);        // dh_hi W_lo
                    umma_tf32_ts(tbase0 + UM_COL_DU, a_hi, bh, idesc_b, 1);        // dh_hi W_hi
                }
                asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar + 8 + 8 * (c & 1)) : "memory");
            }
        }
        // the commits not yet waited for: those of the last two chunks (one if there is a single chunk); after them dU, dQ are complete
        {
            const int nch = HP / 16;
            for (int c = max(nch - 2, 0); c < nch; ++c) {
                ok = ok && mbar_wait(bar + 8 + 8 * (c & 1), phc[c & 1]);
                phc[c & 1] ^= 1;
            }
        }
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        // 4. outputs
        if (ok) {
            float du[32], dq[32];
            tmem_ld16(tbase + UM_COL_DU, reinterpret_cast<float (&)[16]>(du[0]));
            tmem_ld16(tbase + UM_COL_DU + 16, reinterpret_cast<float (&)[16]>(du[16]));
            tmem_ld16(tbase + UM_COL_DQ, reinterpret_cast<float (&)[16]>(dq[0]));
            tmem_ld16(tbase + UM_COL_DQ + 16, reinterpret_cast<float (&)[16]>(dq[16]));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (live) {
                const float Uv = U - b1U, qv = q - b1q;
                Ui[p] = Uv; qraw[p] = qv;
                accU += (double)Uv; accQ += (double)qv;
#pragma unroll
                for (int v = 0; v < ND; ++v) { FpU[(int64_t)v * N + p] = du[v]; FpQ[(int64_t)v * N + p] = dq[v]; }
            }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        ok = __syncthreads_and(ok);                    // all TMEM reads of this tile are done before the next tile overwrites;
                                                       // the whole block leaves the tile loop together after a time-out
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    }
    if (!ok) atomicOr(&flags[FLAG_TENSOR_TIMEOUT], 1);
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(sh_tmem), "n"(UM_COLS));
    const double su = block_sum(accU, sh_red);
    const double sq = block_sum(accQ, sh_red);
    if (threadIdx.x == 0) { atomicAdd(&sums[SUM_E_NEP], su); atomicAdd(&sums[SUM_Q], sq); }
}

// One atom per thread, scalar FMAs: the form used when the 4-/5-body terms are on (35 descriptors; two atoms per thread
// would need 3 x 35 register pairs).
template <int NDT>
__global__ void __launch_bounds__(128)
k_nn1(int64_t N, int T, int H, int nn_stride, const float* __restrict__ nnw, float b1U, float b1q,
      const float4* __restrict__ xyzt, const float* __restrict__ D, float* __restrict__ Ui, float* __restrict__ qraw,
      float* __restrict__ FpU, float* __restrict__ FpQ, double* __restrict__ sums)
{
    constexpr int WP = (NDT + 3) / 4 * 4;
    extern __shared__ __align__(16) float sh_w[];
    __shared__ double sh_red[32];
    {
        const float4* src = reinterpret_cast<const float4*>(nnw);
        float4* dst = reinterpret_cast<float4*>(sh_w);
        for (int i = threadIdx.x; i < T * nn_stride / 4; i += blockDim.x) dst[i] = src[i];
    }
    __syncthreads();
    double accU = 0.0, accQ = 0.0;
    for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < N; p += (int64_t)gridDim.x * blockDim.x) {
        const int ti = __float_as_int(xyzt[p].w);
        const float* w = sh_w + ti * nn_stride;
        const float* b0 = w + H * WP;
        const float* w1U = b0 + H;
        const float* w1q = w1U + H;
        float x[WP], dU[WP], dQ[WP];
#pragma unroll
        for (int v = 0; v < WP; ++v) { x[v] = v < NDT ? D[(int64_t)v * N + p] : 0.f; dU[v] = 0.f; dQ[v] = 0.f; }
        float U = 0.f, q = 0.f;
        for (int mu = 0; mu < H; ++mu) {
            const float4* row = reinterpret_cast<const float4*>(w + mu * WP);
            float wr[WP];
#pragma unroll
            for (int v4 = 0; v4 < WP / 4; ++v4) {
                const float4 t = row[v4];
                wr[4 * v4] = t.x; wr[4 * v4 + 1] = t.y; wr[4 * v4 + 2] = t.z; wr[4 * v4 + 3] = t.w;
            }
            float z0 = -b0[mu], z1 = 0.f;
#pragma unroll
            for (int v = 0; v < NDT; v += 2) { z0 = fmaf(wr[v], x[v], z0); if (v + 1 < NDT) z1 = fmaf(wr[v + 1], x[v + 1], z1); }
            const float hmu = tanh_f32(z0 + z1);
            const float a = w1U[mu], b = w1q[mu];
            U = fmaf(a, hmu, U);
            q = fmaf(b, hmu, q);
            const float dh = fmaf(-hmu, hmu, 1.f);
            const float au = a * dh, bq = b * dh;
#pragma unroll
            for (int v = 0; v < NDT; ++v) { dU[v] = fmaf(au, wr[v], dU[v]); dQ[v] = fmaf(bq, wr[v], dQ[v]); }
        }
        U -= b1U;
        q -= b1q;
        Ui[p] = U;
        qraw[p] = q;
#pragma unroll
        for (int v = 0; v < NDT; ++v) { FpU[(int64_t)v * N + p] = dU[v]; FpQ[(int64_t)v * N + p] = dQ[v]; }
        accU += (double)U;
        accQ += (double)q;
    }
    const double su = block_sum(accU, sh_red);
    const double sq = block_sum(accQ, sh_red);
    if (threadIdx.x == 0) { atomicAdd(&sums[SUM_E_NEP], su); atomicAdd(&sums[SUM_Q], sq); }
}

// a5: Eq. 33 (reading G3): q_i = q_i^raw + (Q - sum_j q_j^raw) / N
__global__ void k_neutralise(int64_t N, const float* __restrict__ qraw, const double* __restrict__ sums, double Qtot,
                             const int* __restrict__ sidx, const int* __restrict__ cm, float* __restrict__ q,
                             int2* __restrict__ qcm, double* __restrict__ charges_out)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const double shift = (Qtot - sums[SUM_Q]) / (double)N;
    const double v = (double)qraw[p] + shift;
    q[p] = (float)v;
    qcm[cm[p]] = make_int2((int)p, __float_as_int((float)v));      // the same charge in the order of the PPPM kernels
    if (charges_out) charges_out[sidx[p]] = v;
}

// ------------------------------------------------------------------------------------------
// a11 (angular part): F_ij = sum_{n,lm} Q_nlm d/dr_ij [ g_n(r_ij) b_lm(rhat_ij) ],
//   Q_nlm = dE/dA_nlm = 2 C_lm Fp_{nl} A_nlm.  With G_lm = sum_n Q_nlm g_n, G'_lm = sum_n Q_nlm g_n':
//   F_ij = rhat sum_lm G'_lm b_lm + [v - (rhat.v) rhat] / r,  v = sum_lm G_lm grad_u b_lm.
// Own sums go to Fa (3 per atom; BEC: 9 per atom = 1/2 r_ij (x) c_ij), pair vectors to f12.
// ------------------------------------------------------------------------------------------
// ATOMV (with VIRIAL, not BEC): the pair term -r_ij (x) F_ij belongs to the per-atom virial of atom j (Eq. 12:
// W_j = sum_i r_ji (x) F_ij) and is scattered to rows 3..11 of Facc.
template <int T, bool BEC, bool VIRIAL, bool ATOMV = false, bool ZBL = false>
#ifndef QNEP_FA_VIR_BLOCKS
#define QNEP_FA_VIR_BLOCKS 4
#endif
#ifndef QNEP_FA_BLOCKS
#define QNEP_FA_BLOCKS 4
#endif
__global__ void __launch_bounds__(ANG_BLOCK, BEC || ATOMV ? 4 : (VIRIAL ? QNEP_FA_VIR_BLOCKS : QNEP_FA_BLOCKS))
k_force_angular(int64_t N, const float4* __restrict__ xyzt, const float4* __restrict__ lvA, int capLA, const int* __restrict__ nlvA,
                const float* __restrict__ cA, const float* __restrict__ cR, float rcinv, const float* __restrict__ FpU,
                const float* __restrict__ FpQ, const float* __restrict__ phi, float sqrt_eps, const float* __restrict__ Ain,
                float* __restrict__ Fp, float* __restrict__ recA, float4* __restrict__ recB, float* __restrict__ Facc,
                double* __restrict__ sums, ZblParams zbl, int hb /* 4-/5-body terms on */)
{
    // Packed angular coefficient table for the loop below: row (ti, tj, n) holds ten float2,
    //   [0] = (2 c_0 + sum_{k>=1} c_k, 0)  and  [k] = (c_k, k c_k), k = 1..8   ([9] is padding),
    // so that  (sum_k c_k (T_k + 1), sum_k c_k k U_{k-1}) = [0] + sum_{k>=1} [k] * (T_k, U_{k-1})  in eight packed FMAs.
    __shared__ __align__(16) float2 sh_c2[T * T * NR * FA_KP2];
    __shared__ __align__(16) float sh_cR[T * T * NR * KP];
    __shared__ float4 sh_ring[ANG_DEPTH][ANG_BLOCK];
    __shared__ double sh_red[32];
    for (int i = threadIdx.x; i < T * T * NR * KP; i += blockDim.x) sh_cR[i] = cR[i];
    for (int i = threadIdx.x; i < T * T * NR; i += blockDim.x) {
        const float* c = cA + i * KP;
        float c0 = 2.f * c[0];
#pragma unroll
        for (int k = 1; k < NB; ++k) { c0 += c[k]; sh_c2[i * FA_KP2 + k] = make_float2(c[k], (float)k * c[k]); }
        sh_c2[i * FA_KP2] = make_float2(c0, 0.f);
        sh_c2[i * FA_KP2 + 9] = make_float2(0.f, 0.f);
    }
    __syncthreads();
    const int tid = threadIdx.x;
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + tid;
    float W[9];
#pragma unroll
    for (int a = 0; a < 9; ++a) W[a] = 0.f;
    if (p < N) {
        const int n = nlvA[p];
        const float4* rows = lvA + qnep_tiled_base(p, capLA);
#pragma unroll
        for (int k = 0; k < ANG_DEPTH; ++k) {
            if (k < n) cp_async16_cg(&sh_ring[k][tid], rows + (int64_t)k * QNEP_TILE);
            cp_async_commit();
        }
        const float4 xi = xyzt[p];
        const int ti = __float_as_int(xi.w);
        // a10: Fp = dU/dD + phi_eff dq/dD (S6: phi_eff = phi - mean phi); BEC mode: Fp = sqrt(eps_inf) dq/dD (Eq. 24, 28; S12).
        // The radial part goes into the gather records of the radial force kernel, one per species t of the atom
        // that will read it: recA[t][p] = (x, y, z, P^t_0..P^t_4), recB[t][p] = (P^t_5..P^t_8), P^t_k = sum_n Fp_n c^{ti t}_{nk}.
        float cu, cq;
        if (BEC) { cu = 0.f; cq = sqrt_eps; }
        else { cu = 1.f; cq = phi[p] - (float)(sums[SUM_PHI] / (double)N); }
        {
            float fr[NR];
#pragma unroll
            for (int v = 0; v < NR; ++v) {
                fr[v] = cu * FpU[(int64_t)v * N + p] + cq * FpQ[(int64_t)v * N + p];
                Fp[(int64_t)v * N + p] = fr[v];
            }
#pragma unroll
            for (int t = 0; t < T; ++t) {
                float pk[NB];
#pragma unroll
                for (int k = 0; k < NB; ++k) {
                    float v = 0.f;
#pragma unroll
                    for (int a = 0; a < NR; ++a) v = fmaf(fr[a], sh_cR[((ti * T + t) * NR + a) * KP + k], v);
                    pk[k] = v;
                }
                float4* r4 = reinterpret_cast<float4*>(recA + 8 * ((int64_t)t * N + p));
                r4[0] = make_float4(xi.x, xi.y, xi.z, pk[0]);
                r4[1] = make_float4(pk[1], pk[2], pk[3], pk[4]);
                recB[(int64_t)t * N + p] = make_float4(pk[5], pk[6], pk[7], pk[8]);
            }
        }
        // Q_nlm = dE/dA_nlm = 2 C_lm Fp_nl A_nlm, held as register PAIRS in the order of c_fa_pair (two harmonics with
        // the same zero pattern of their gradient share a pair): the loop below is bound by issue slots, and a packed
        // FMA (FFMA2) does two FP32 FMAs per issued instruction.
        float2 Q2[NR][NLM / 2];
#pragma unroll
        for (int a = 0; a < NR; ++a) {
            float fpl[4];
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                const int64_t v = NR + a * 4 + l;
                const float val = cu * FpU[v * N + p] + cq * FpQ[v * N + p];
                Fp[v * N + p] = val;
                fpl[l] = 2.f * val;
            }
            // higher-body terms (reading Z2): dE/dA_lm for lm = 0..7 from q5 = (w.w)^2 and q4 = tr(T^3), S = T^2:
            //   d q5 / d A_{0,1,2} = 4 (w.w) A;   d q4 / d A_3..7 = S_zz - (S_xx + S_yy)/2, 6 S_xz, 6 S_yz, 3/2 (S_xx - S_yy), 3 S_xy
            float extra[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
            if (hb) {
                const int64_t v4 = ND + a, v5 = ND + NR + a;
                const float f4 = cu * FpU[v4 * N + p] + cq * FpQ[v4 * N + p], f5 = cu * FpU[v5 * N + p] + cq * FpQ[v5 * N + p];
                Fp[v4 * N + p] = f4; Fp[v5 * N + p] = f5;
                float A8[8], Tn[6], Sn[6], w2;
#pragma unroll
                for (int lm = 0; lm < 8; ++lm) A8[lm] = Ain[(int64_t)(a * NLM + lm) * N + p];
                hb_moments(A8, Tn, Sn, w2);
                const float c5 = 4.f * w2 * f5;
                extra[0] = c5 * A8[0]; extra[1] = c5 * A8[1]; extra[2] = c5 * A8[2];
                extra[3] = f4 * (Sn[2] - 0.5f * (Sn[0] + Sn[1]));
                extra[4] = 6.f * f4 * Sn[4]; extra[5] = 6.f * f4 * Sn[5];
                extra[6] = 1.5f * f4 * (Sn[0] - Sn[1]); extra[7] = 3.f * f4 * Sn[3];
            }
#pragma unroll
            for (int m = 0; m < NLM / 2; ++m) {
                constexpr int pa[NLM / 2] = {0, 8, 1, 6, 13, 22, 4, 9, 11, 16, 18, 20};
                constexpr int pb[NLM / 2] = {3, 15, 2, 7, 14, 23, 5, 10, 12, 17, 19, 21};
                Q2[a][m] = make_float2(c_Clm[pa[m]] * fpl[l_of_lm(pa[m])] * Ain[(int64_t)(a * NLM + pa[m]) * N + p] + (pa[m] < 8 ? extra[pa[m]] : 0.f),
                                       c_Clm[pb[m]] * fpl[l_of_lm(pb[m])] * Ain[(int64_t)(a * NLM + pb[m]) * N + p] + (pb[m] < 8 ? extra[pb[m]] : 0.f));
            }
        }
        float Fx = 0.f, Fy = 0.f, Fz = 0.f;
        for (int s = 0; s < n; ++s) {
            cp_async_wait<ANG_DEPTH - 1>();
            const float4 pr = sh_ring[s & (ANG_DEPTH - 1)][tid];
            if (s + ANG_DEPTH < n) cp_async16_cg(&sh_ring[s & (ANG_DEPTH - 1)][tid], rows + (int64_t)(s + ANG_DEPTH) * QNEP_TILE);
            cp_async_commit();
            const float dx = pr.x, dy = pr.y, dz = pr.z;
            const float r2 = dx * dx + dy * dy + dz * dz;
            const float rinv = fast_rsqrt(r2), r = r2 * rinv;
            const int jw = __float_as_int(pr.w);
            const int j = jw & QNEP_NL_MASK;
            // g_n = 1/2 fc sum_k c_nk (T_k + 1),  g_n' = A sum_k c_nk k U_{k-1} + B sum_k c_nk (T_k + 1)   (see ChebDeriv);
            // V_k = (T_k, U_{k-1}) obeys V_{k+1} = 2x V_k - V_{k-1} in both components
            float2 g2[NR], dg2[NR];
            {
                const float t = r * rcinv;
                float sn, cs;
                __sincosf(3.14159265358979f * t, &sn, &cs);
                const float tm1 = t - 1.f;
                const float xx = 2.f * tm1 * tm1 - 1.f;
                const float hfc = 0.25f + 0.25f * cs;
                const float cA_ = hfc * (4.f * tm1 * rcinv);
                const float cB_ = -0.7853981633974483f * rcinv * sn;
                const float2 x22 = make_float2(xx + xx, xx + xx);
                float2 V[NB];
                V[0] = make_float2(1.f, 0.f);
                V[1] = make_float2(xx, 1.f);
#pragma unroll
                for (int k = 2; k < NB; ++k) V[k] = __ffma2_rn(x22, V[k - 1], make_float2(-V[k - 2].x, -V[k - 2].y));
                const float4* c4 = reinterpret_cast<const float4*>(sh_c2 + (ti * T + (int)((unsigned)jw >> QNEP_NL_SHIFT)) * NR * FA_KP2);
#pragma unroll
                for (int a = 0; a < NR; ++a) {
                    const float4 q0 = c4[a * 5], q1 = c4[a * 5 + 1], q2 = c4[a * 5 + 2], q3 = c4[a * 5 + 3], q4 = c4[a * 5 + 4];
                    float2 acc = make_float2(q0.x, q0.y);
                    acc = __ffma2_rn(make_float2(q0.z, q0.w), V[1], acc);
                    acc = __ffma2_rn(make_float2(q1.x, q1.y), V[2], acc);
                    acc = __ffma2_rn(make_float2(q1.z, q1.w), V[3], acc);
                    acc = __ffma2_rn(make_float2(q2.x, q2.y), V[4], acc);
                    acc = __ffma2_rn(make_float2(q2.z, q2.w), V[5], acc);
                    acc = __ffma2_rn(make_float2(q3.x, q3.y), V[6], acc);
                    acc = __ffma2_rn(make_float2(q3.z, q3.w), V[7], acc);
                    acc = __ffma2_rn(make_float2(q4.x, q4.y), V[8], acc);
                    const float gv = hfc * acc.x, dgv = fmaf(cA_, acc.y, cB_ * acc.x);
                    g2[a] = make_float2(gv, gv);
                    dg2[a] = make_float2(dgv, dgv);
                }
            }
            const float x = dx * rinv, y = dy * rinv, z = dz * rinv;
            const float x2 = x * x, y2 = y * y, z2 = z * z, xy = x * y, xz = x * z, yz = y * z;
            const float x2my2 = x2 - y2;
            float2 s02 = make_float2(0.f, 0.f), vx2 = s02, vy2 = s02, vz2 = s02;
            float vxs = 0.f, vys = 0.f;
            // G_lm = sum_n Q_nlm g_n, G'_lm = sum_n Q_nlm g_n' for the pair m; then s0 += G' b, v += G grad b
#define QNEP_HPAIR(M)                                                                   \
            float2 G_ = __fmul2_rn(Q2[0][M], g2[0]), Gp_ = __fmul2_rn(Q2[0][M], dg2[0]);  \
            _Pragma("unroll") for (int a = 1; a < NR; ++a) {                             \
                G_ = __ffma2_rn(Q2[a][M], g2[a], G_);                                    \
                Gp_ = __ffma2_rn(Q2[a][M], dg2[a], Gp_);                                 \
            }
            const float f5 = 5.f * z2 - 1.f;
            const float t3 = 3.f * x2my2;            // 3x^2 - 3y^2
            const float f7 = 7.f * z2 - 1.f, f73 = 7.f * z2 - 3.f;
            const float cx = (x2 - 3.f * y2) * x, cy = (3.f * x2 - y2) * y;   // x^3 - 3xy^2, 3x^2 y - y^3
            {   // (0, 3): z | 3z^2 - 1; gradients along z only
                QNEP_HPAIR(0)
                s02 = __ffma2_rn(Gp_, make_float2(z, 3.f * z2 - 1.f), s02);
                vz2 = __ffma2_rn(G_, make_float2(1.f, 6.f * z), vz2);
            }
            {   // (8, 15): (5z^2 - 3) z | (35z^2 - 30) z^2 + 3; gradients along z only
                QNEP_HPAIR(1)
                s02 = __ffma2_rn(Gp_, make_float2((5.f * z2 - 3.f) * z, (35.f * z2 - 30.f) * z2 + 3.f), s02);
                vz2 = __ffma2_rn(G_, make_float2(15.f * z2 - 3.f, (140.f * z2 - 60.f) * z), vz2);
            }
            {   // (1, 2): x | y
                QNEP_HPAIR(2)
                s02 = __ffma2_rn(Gp_, make_float2(x, y), s02);
                vxs += G_.x; vys += G_.y;
            }
            {   // (6, 7): x^2 - y^2 | 2xy
                QNEP_HPAIR(3)
                s02 = __ffma2_rn(Gp_, make_float2(x2my2, 2.f * xy), s02);
                vx2 = __ffma2_rn(G_, make_float2(2.f * x, 2.f * y), vx2);
                vy2 = __ffma2_rn(G_, make_float2(-2.f * y, 2.f * x), vy2);
            }
            {   // (13, 14): x^3 - 3xy^2 | 3x^2 y - y^3
                QNEP_HPAIR(4)
                s02 = __ffma2_rn(Gp_, make_float2(cx, cy), s02);
                vx2 = __ffma2_rn(G_, make_float2(t3, 6.f * xy), vx2);
                vy2 = __ffma2_rn(G_, make_float2(-6.f * xy, t3), vy2);
            }
            {   // (22, 23): (x^2 - y^2)^2 - 4x^2 y^2 | 4 (x^2 - y^2) xy
                QNEP_HPAIR(5)
                s02 = __ffma2_rn(Gp_, make_float2(x2my2 * x2my2 - 4.f * x2 * y2, 4.f * x2my2 * xy), s02);
                vx2 = __ffma2_rn(G_, make_float2(4.f * cx, 4.f * cy), vx2);
                vy2 = __ffma2_rn(G_, make_float2(-4.f * cy, 4.f * cx), vy2);
            }
            {   // (4, 5): xz | yz
                QNEP_HPAIR(6)
                s02 = __ffma2_rn(Gp_, make_float2(xz, yz), s02);
                vxs = fmaf(G_.x, z, vxs); vys = fmaf(G_.y, z, vys);
                vz2 = __ffma2_rn(G_, make_float2(x, y), vz2);
            }
            {   // (9, 10): (5z^2 - 1) x | (5z^2 - 1) y
                QNEP_HPAIR(7)
                s02 = __ffma2_rn(Gp_, make_float2(f5 * x, f5 * y), s02);
                vxs = fmaf(G_.x, f5, vxs); vys = fmaf(G_.y, f5, vys);
                vz2 = __ffma2_rn(G_, make_float2(10.f * xz, 10.f * yz), vz2);
            }
            {   // (11, 12): (x^2 - y^2) z | 2xyz
                QNEP_HPAIR(8)
                s02 = __ffma2_rn(Gp_, make_float2(x2my2 * z, 2.f * xy * z), s02);
                vx2 = __ffma2_rn(G_, make_float2(2.f * xz, 2.f * yz), vx2);
                vy2 = __ffma2_rn(G_, make_float2(-2.f * yz, 2.f * xz), vy2);
                vz2 = __ffma2_rn(G_, make_float2(x2my2, 2.f * xy), vz2);
            }
            {   // (16, 17): (7z^2 - 3) xz | (7z^2 - 3) yz
                QNEP_HPAIR(9)
                const float f73z = f73 * z, g21 = 21.f * z2 - 3.f;
                s02 = __ffma2_rn(Gp_, make_float2(f73 * xz, f73 * yz), s02);
                vxs = fmaf(G_.x, f73z, vxs); vys = fmaf(G_.y, f73z, vys);
                vz2 = __ffma2_rn(G_, make_float2(g21 * x, g21 * y), vz2);
            }
            {   // (18, 19): (7z^2 - 1)(x^2 - y^2) | (7z^2 - 1) 2xy
                QNEP_HPAIR(10)
                const float xf7 = 2.f * x * f7, yf7 = 2.f * y * f7;
                s02 = __ffma2_rn(Gp_, make_float2(f7 * x2my2, f7 * 2.f * xy), s02);
                vx2 = __ffma2_rn(G_, make_float2(xf7, yf7), vx2);
                vy2 = __ffma2_rn(G_, make_float2(-yf7, xf7), vy2);
                vz2 = __ffma2_rn(G_, make_float2(14.f * z * x2my2, 28.f * xy * z), vz2);
            }
            {   // (20, 21): (x^3 - 3xy^2) z | (3x^2 y - y^3) z
                QNEP_HPAIR(11)
                const float t3z = t3 * z, xyz6 = 6.f * xy * z;
                s02 = __ffma2_rn(Gp_, make_float2(cx * z, cy * z), s02);
                vx2 = __ffma2_rn(G_, make_float2(t3z, xyz6), vx2);
                vy2 = __ffma2_rn(G_, make_float2(-xyz6, t3z), vy2);
                vz2 = __ffma2_rn(G_, make_float2(cx, cy), vz2);
            }
#undef QNEP_HPAIR
            float s0 = s02.x + s02.y;
            if (!BEC && ZBL && r2 < zbl.r2sq) {
                // ZBL site energy 1/2 sum_j U(r_ij): partial force 1/2 U'(r_ij) rhat_ij, booked like the NEP ones (reading Z1)
                float u, du;
                qnep_zbl_eval(zbl, ti, (int)((unsigned)jw >> QNEP_NL_SHIFT), r, rinv, u, du);
                s0 = fmaf(0.5f, du, s0);
            }
            const float vx = vxs + (vx2.x + vx2.y), vy = vys + (vy2.x + vy2.y), vz = vz2.x + vz2.y;
            const float uv = x * vx + y * vy + z * vz;
            const float fx = s0 * x + (vx - uv * x) * rinv;
            const float fy = s0 * y + (vy - uv * y) * rinv;
            const float fz = s0 * z + (vz - uv * z) * rinv;
            if (BEC) {
                // Z_i += 1/2 r_ij (x) c_ij ;  Z_j += 1/2 r_ji (x) c_ij = -1/2 r_ij (x) c_ij   (Eq. 28)
                const float hx = 0.5f * dx, hy = 0.5f * dy, hz = 0.5f * dz;
                const float z9[9] = {hx * fx, hx * fy, hx * fz, hy * fx, hy * fy, hy * fz, hz * fx, hz * fy, hz * fz};
#pragma unroll
                for (int a = 0; a < 9; ++a) { W[a] += z9[a]; atomicAdd(&Facc[(int64_t)a * N + j], -z9[a]); }
            } else {
                // F_i += F_ij, F_j -= F_ij (Eq. 11)
                Fx += fx; Fy += fy; Fz += fz;
                atomicAdd(&Facc[j], -fx); atomicAdd(&Facc[N + j], -fy); atomicAdd(&Facc[2 * N + j], -fz);
                if (VIRIAL) {   // -r_ij (x) F_ij (Eq. 12)
                    W[0] = fmaf(dx, fx, W[0]); W[1] = fmaf(dx, fy, W[1]); W[2] = fmaf(dx, fz, W[2]);
                    W[3] = fmaf(dy, fx, W[3]); W[4] = fmaf(dy, fy, W[4]); W[5] = fmaf(dy, fz, W[5]);
                    W[6] = fmaf(dz, fx, W[6]); W[7] = fmaf(dz, fy, W[7]); W[8] = fmaf(dz, fz, W[8]);
                }
                if (ATOMV) {
                    const float w9[9] = {dx * fx, dx * fy, dx * fz, dy * fx, dy * fy, dy * fz, dz * fx, dz * fy, dz * fz};
#pragma unroll
                    for (int a = 0; a < 9; ++a) atomicAdd(&Facc[(int64_t)(3 + a) * N + j], -w9[a]);
                }
            }
        }
        if (BEC) {
#pragma unroll
            for (int a = 0; a < 9; ++a) atomicAdd(&Facc[(int64_t)a * N + p], W[a]);
        } else {
            atomicAdd(&Facc[p], Fx); atomicAdd(&Facc[N + p], Fy); atomicAdd(&Facc[2 * N + p], Fz);
        }
    }
    if (!BEC && VIRIAL) {
#pragma unroll
        for (int a = 0; a < 9; ++a) {
            const double w = block_sum((double)W[a], sh_red);
            if (threadIdx.x == 0) atomicAdd(&sums[SUM_COUNT + (blockIdx.x % QNEP_WSTRIPES) * QNEP_WSTRIDE + a], -w);
        }
    }
}

// ------------------------------------------------------------------------------------------
// a11 (radial part + assembly): F_i = sum_j (s_ij + s_ji) rhat_ij  +  angular accumulator  +  static electrostatic
//   force;  s_ij = sum_k P^{i,tj}_k f_k'(r_ij),  s_ji = sum_k P^{j,ti}_k f_k'(r_ij),  P^{i,t}_k = sum_n Fp^i_n c^{ti t}_{nk}.
// BEC mode (a12): Z_i = qt_i I + 1/2 sum_j r_ij (x) (c_ij + c_ji).
// Per neighbour two gathers from the records the angular kernel wrote for readers of species ti: recA[ti][j] =
// (x, y, z, P_0..P_4) (one 32-byte sector, LDG.256) and recB[ti][j] = (P_5..P_8).  The list is type-major, so the
// thread's own vector P^{i,tj} changes T - 1 times along the list (it is the thread's own record for species tj).
// List words run through a cp.async ring RAD_DW rows ahead, records through a register ring RAD_DX deep.
// Output in ORIGINAL atom order, float64.
// ------------------------------------------------------------------------------------------
constexpr int RAD_BLOCK = 128, RAD_LV = 4;      // list vectors (4 slots each) in flight; records are requested 4 slots ahead

__device__ __forceinline__ void ldg256(const float* p, float (&v)[8])
{
    asm volatile("ld.global.nc.v8.f32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "l"(p));
}

// ATOMV (with VIRIAL): per-atom virial W_i = sum_j r_ij (x) F_ji with the radial F_ji = -s_ji rhat_ij, plus the angular
// terms scattered by k_force_angular (Facc rows 3..11) and the static electrostatic parts (Wat), to atomv_out [9][N].
// (launch bounds: 128 registers at four blocks per SM; forcing 5 or 6 blocks spills: 0.61 -> 0.83 / 1.31 ms)
template <int T, bool BEC, bool VIRIAL, bool ATOMV = false>
__global__ void __launch_bounds__(RAD_BLOCK)
k_force_radial(int64_t N, Geometry g, const float* __restrict__ recA, const float4* __restrict__ recB,
               const float4* __restrict__ xyzt, const int4* __restrict__ lvR, int capLR, const int* __restrict__ nlvR,
               const int* __restrict__ lvRend, float rcinv, const float* __restrict__ Facc, const float* __restrict__ Fs,
               const float* __restrict__ q, float sqrt_eps, const int* __restrict__ sidx, double* __restrict__ out,
               double* __restrict__ sums, const float* __restrict__ Wat, double* __restrict__ atomv_out)
{
    __shared__ int4 sh_w[RAD_LV][RAD_BLOCK];
    __shared__ double sh_red[32];
    const CellVecs cv = qnep_cell_vecs(g.cellv, g.triclinic);
    const int tid = threadIdx.x;
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + tid;
    float W[9];
    float Wa[ATOMV ? 9 : 1];
#pragma unroll
    for (int a = 0; a < 9; ++a) W[a] = 0.f;
#pragma unroll
    for (int a = 0; a < (ATOMV ? 9 : 1); ++a) Wa[a] = 0.f;
    if (p < N) {
        const int n = nlvR[p];
        const int n4 = (n + 3) >> 2;
        const int4* vbase = lvR + qnep_tiled_base(p, capLR / 4);
        const float4 xi = xyzt[p];
        const int ti = __float_as_int(xi.w);
        const float* gA = recA + 8 * (int64_t)ti * N;       // records for readers of my species
        const float4* gB = recB + (int64_t)ti * N;
        // prologue: vector 0 by a plain load (its records are requested at once), vectors 1..LV through the ring.
        // cp.async groups: LV in the prologue, one per iteration; at the top of iteration v the group of vector v + 1
        // is number v + 1 of LV + v, so LV - 1 may stay pending.
        int4 cur = n > 0 ? vbase[0] : make_int4((int)p, (int)p, (int)p, (int)p);
#pragma unroll
        for (int k = 1; k <= RAD_LV; ++k) {
            if (k < n4) cp_async16_cg(&sh_w[k & (RAD_LV - 1)][tid], vbase + (int64_t)k * QNEP_TILE);
            cp_async_commit();
        }
        float ra[4][8];
        float4 rb[4];
        {
            const int e0[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int j = u < n ? (e0[u] & QNEP_NL_MASK) : (int)p;
                ldg256(gA + 8 * (int64_t)j, ra[u]);
                rb[u] = __ldg(gB + j);
            }
        }
        int tj = -1, seg_end = 0;
        float Pi[NB];
#pragma unroll
        for (int k = 0; k < NB; ++k) Pi[k] = 0.f;
        float Fx = 0.f, Fy = 0.f, Fz = 0.f;
        for (int v = 0; v < n4; ++v) {
            cp_async_wait<RAD_LV - 1>();
            int4 nxt = cur;
            if (v + 1 < n4) nxt = sh_w[(v + 1) & (RAD_LV - 1)][tid];
            if (v + 1 + RAD_LV < n4) cp_async16_cg(&sh_w[(v + 1) & (RAD_LV - 1)][tid], vbase + (int64_t)(v + 1 + RAD_LV) * QNEP_TILE);
            cp_async_commit();
            const int ec[4] = {cur.x, cur.y, cur.z, cur.w};
            const int en[4] = {nxt.x, nxt.y, nxt.z, nxt.w};
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int s = 4 * v + u;
                if (s < n) {
                    const int e = ec[u];
                    const float (&a8)[8] = ra[u];
                    const float4& b4 = rb[u];
                    if (s >= seg_end) {
                        // next non-empty species segment: my own vector for neighbours of species tj is my record for tj
                        do { ++tj; seg_end = lvRend[(int64_t)tj * N + p]; } while (s >= seg_end && tj < T - 1);
                        float o8[8];
                        ldg256(recA + 8 * ((int64_t)tj * N + p), o8);
                        const float4 o4 = __ldg(recB + (int64_t)tj * N + p);
                        Pi[0] = o8[3]; Pi[1] = o8[4]; Pi[2] = o8[5]; Pi[3] = o8[6]; Pi[4] = o8[7];
                        Pi[5] = o4.x; Pi[6] = o4.y; Pi[7] = o4.z; Pi[8] = o4.w;
                    }
                    float dx = a8[0] - xi.x, dy = a8[1] - xi.y, dz = a8[2] - xi.z;
                    qnep_add_image_shift(e, cv, dx, dy, dz);
                    const float r2 = dx * dx + dy * dy + dz * dz;
                    const float rinv = fast_rsqrt(r2), r = r2 * rinv;
                    ChebDeriv cd;
                    cd.eval(r, rcinv);
                    const float Pj[NB] = {a8[3], a8[4], a8[5], a8[6], a8[7], b4.x, b4.y, b4.z, b4.w};
                    float sij, sji;
                    if (BEC || ATOMV) {
                        sij = cd.dot(Pi);
                        sji = cd.dot(Pj);
                    } else {
                        // only s_ij + s_ji is needed: one contraction with P^{i,tj} + P^{j,ti}.  That holds for the TOTAL
                        // virial too: sum_i sum_j r_ij (x) rhat_ij s_ij runs over ordered pairs, and the terms (i, j) and
                        // (j, i) have the same dyad r_ij (x) rhat_ij, so every atom may book 1/2 (s_ij + s_ji) instead of s_ij.
                        const float2 Pp[4] = {__fadd2_rn(make_float2(Pi[1], Pi[2]), make_float2(a8[4], a8[5])),
                                              __fadd2_rn(make_float2(Pi[3], Pi[4]), make_float2(a8[6], a8[7])),
                                              __fadd2_rn(make_float2(Pi[5], Pi[6]), make_float2(b4.x, b4.y)),
                                              __fadd2_rn(make_float2(Pi[7], Pi[8]), make_float2(b4.z, b4.w))};
                        sij = 0.5f * cd.dot_pairs(Pi[0] + a8[3], Pp);
                        sji = sij;
                    }
                    const float ux = dx * rinv, uy = dy * rinv, uz = dz * rinv;
                    if (BEC) {
                        // 1/2 r_ij (x) (c_ij + c_ji), c_ij = s_ij rhat, c_ji = s_ji rhat_ji = -s_ji rhat
                        const float w = 0.5f * (sij - sji);
                        W[0] = fmaf(dx, w * ux, W[0]); W[1] = fmaf(dx, w * uy, W[1]); W[2] = fmaf(dx, w * uz, W[2]);
                        W[3] = fmaf(dy, w * ux, W[3]); W[4] = fmaf(dy, w * uy, W[4]); W[5] = fmaf(dy, w * uz, W[5]);
                        W[6] = fmaf(dz, w * ux, W[6]); W[7] = fmaf(dz, w * uy, W[7]); W[8] = fmaf(dz, w * uz, W[8]);
                    } else {
                        const float w = sij + sji;
                        Fx = fmaf(w, ux, Fx); Fy = fmaf(w, uy, Fy); Fz = fmaf(w, uz, Fz);
                        if (VIRIAL) {
                            const float wx = sij * ux, wy = sij * uy, wz = sij * uz;     // F_ij
                            W[0] = fmaf(dx, wx, W[0]); W[1] = fmaf(dx, wy, W[1]); W[2] = fmaf(dx, wz, W[2]);
                            W[3] = fmaf(dy, wx, W[3]); W[4] = fmaf(dy, wy, W[4]); W[5] = fmaf(dy, wz, W[5]);
                            W[6] = fmaf(dz, wx, W[6]); W[7] = fmaf(dz, wy, W[7]); W[8] = fmaf(dz, wz, W[8]);
                        }
                        if (ATOMV) {
                            const float ax = -sji * ux, ay = -sji * uy, az = -sji * uz;  // F_ji = s_ji rhat_ji
                            Wa[0] = fmaf(dx, ax, Wa[0]); Wa[1] = fmaf(dx, ay, Wa[1]); Wa[2] = fmaf(dx, az, Wa[2]);
                            Wa[3] = fmaf(dy, ax, Wa[3]); Wa[4] = fmaf(dy, ay, Wa[4]); Wa[5] = fmaf(dy, az, Wa[5]);
                            Wa[6] = fmaf(dz, ax, Wa[6]); Wa[7] = fmaf(dz, ay, Wa[7]); Wa[8] = fmaf(dz, az, Wa[8]);
                        }
                    }
                    // the record registers are free again: request the record of slot s + 4 into them
                    if (s + 4 < n) {
                        const int j2 = en[u] & QNEP_NL_MASK;
                        ldg256(gA + 8 * (int64_t)j2, ra[u]);
                        rb[u] = __ldg(gB + j2);
                    }
                }
            }
            cur = nxt;
        }
        cp_async_wait<0>();
        const int io = sidx[p];
        if (BEC) {
            const float qt = sqrt_eps * q[p];
#pragma unroll
            for (int a = 0; a < 9; ++a) {
                float v = W[a] + Facc[(int64_t)a * N + p];
                if (a == 0 || a == 4 || a == 8) v += qt;
                out[(int64_t)a * N + io] = (double)v;
            }
        } else {
            out[io] = (double)Fx + (double)Facc[p] + (double)Fs[p];
            out[N + io] = (double)Fy + (double)Facc[N + p] + (double)Fs[N + p];
            out[2 * N + io] = (double)Fz + (double)Facc[2 * N + p] + (double)Fs[2 * N + p];
            if (ATOMV) {
#pragma unroll
                for (int a = 0; a < 9; ++a)
                    atomv_out[(int64_t)a * N + io] = (double)Wa[a] + (double)Facc[(int64_t)(3 + a) * N + p] + (double)Wat[(int64_t)a * N + p];
            }
        }
    }
    if (!BEC && VIRIAL) {
#pragma unroll
        for (int a = 0; a < 9; ++a) {
            const double w = block_sum((double)W[a], sh_red);
            if (threadIdx.x == 0) atomicAdd(&sums[SUM_COUNT + (blockIdx.x % QNEP_WSTRIPES) * QNEP_WSTRIDE + a], -w);
        }
    }
}

// ------------------------------------------------------------------------------------------
// dependent-free FFMA loop: the FP32 roofline denominator measured in the same run
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_fma_peak(int iters, float seed, float* __restrict__ out)
{
    float a[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = seed + (float)(threadIdx.x + i);
    const float m = 0.999999f, c = 1e-7f * seed;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == 123.456f) out[0] = s;     // never true; keeps the loop alive
}

template <typename F>
int dispatch_T(int T, F&& f)
{
    switch (T) {
        case 1: f(std::integral_constant<int, 1>()); return 0;
        case 2: f(std::integral_constant<int, 2>()); return 0;
        case 3: f(std::integral_constant<int, 3>()); return 0;
        case 4: f(std::integral_constant<int, 4>()); return 0;
    }
    return -1;
}

}  // namespace

int qnep_launch_pairs(qnep_handle* h, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + PAIRS_BLOCK - 1) / PAIRS_BLOCK);
    const float rcinv = (float)(1.0 / h->model.rc_r);
    dispatch_T(h->model.n_types, [&](auto t) {
        constexpr int T = decltype(t)::value;
        static bool attr_set = false;                        // one flag per instantiation (the lambda is generic)
        if (!attr_set) {
            cudaFuncSetAttribute(k_pairs<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PAIRS_SMEM);
            cudaFuncSetAttribute(k_pairs<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PAIRS_SMEM);
            attr_set = true;
        }
        auto kern = h->geo.triclinic ? k_pairs<T, true> : k_pairs<T, false>;
        kern<<<nb, PAIRS_BLOCK, PAIRS_SMEM, s>>>(N, h->geo, h->d_xyzt, h->d_nlR, h->d_nnR, h->d_nlRend, h->d_cR, rcinv, h->capR, h->capLR, h->capLA,
                                              h->d_lvR, h->d_nlvR, h->d_lvRend, h->d_lvA, h->d_nlvA, h->d_D, h->d_flags);
    });
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int qnep_launch_desc_angular(qnep_handle* h, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 63) / 64);
    const float rcinv = (float)(1.0 / h->model.rc_a);
    dispatch_T(h->model.n_types, [&](auto t) {
        constexpr int T = decltype(t)::value;
        if (h->zbl.on) k_desc_angular<T, true><<<nb, ANG_BLOCK, 0, s>>>(N, h->d_xyzt, h->d_lvA, h->capLA, h->d_nlvA, h->d_cA, rcinv, h->d_D, h->d_A, h->zbl, h->d_sums, h->ND == QNEP_NDESC_HB ? 1 : 0);
        else k_desc_angular<T, false><<<nb, ANG_BLOCK, 0, s>>>(N, h->d_xyzt, h->d_lvA, h->capLA, h->d_nlvA, h->d_cA, rcinv, h->d_D, h->d_A, h->zbl, h->d_sums, h->ND == QNEP_NDESC_HB ? 1 : 0);
    });
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int qnep_launch_nn(qnep_handle* h, double* charges_out, cudaStream_t s)
{
    const int64_t N = h->N;
    const size_t smem = sizeof(float) * (size_t)h->model.n_types * h->nn_stride;
    static bool attr_set = false;
    static int sms = 0;
    if (!sms) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev); if (sms <= 0) sms = 148; }
    const int nb = (int)std::min<int64_t>((N + 2 * NN_BLOCK - 1) / (2 * NN_BLOCK), (int64_t)sms * QNEP_NN_MINB);      // persistent: QNEP_NN_MINB blocks of 128 threads per SM
    if (!attr_set) {
        QNEP_CUDA_OK(h, cudaFuncSetAttribute(k_nn, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        attr_set = true;
    }
    if (h->ND == QNEP_NDESC && h->nn_tensor == 2) {
        const int HP = (h->model.n_neurons + 15) / 16 * 16;
        const size_t smem_u = sizeof(float) * (size_t)(6 * 32 * HP + 4 * HP);
        static bool attr_u = false;
        if (!attr_u) { QNEP_CUDA_OK(h, cudaFuncSetAttribute(k_nn_umma, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024)); attr_u = true; }
        const int nbu = (int)std::min<int64_t>((N + 127) / 128 + h->model.n_types, (int64_t)sms * 2);
        k_nn_umma<<<nbu, 128, smem_u, s>>>(N, h->model.n_types, h->model.n_neurons, HP, h->nn_stride, h->d_nn, h->b1U, h->b1q, h->d_start,
                                           h->geo.ncells, h->d_D, h->d_Ui, h->d_qraw, h->d_FpU, h->d_FpQ, h->d_sums, h->d_flags);
    } else if (h->ND == QNEP_NDESC && h->nn_tensor == 1) {
        const int HP = (h->model.n_neurons + 7) / 8 * 8;
        const size_t smem_t = sizeof(float) * (size_t)h->model.n_types * (2 * HP * NNM_LD + 3 * HP);
        static bool attr_t = false;
        if (!attr_t) { QNEP_CUDA_OK(h, cudaFuncSetAttribute(k_nn_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)); attr_t = true; }
        const int nbt = (int)std::min<int64_t>((N + 127) / 128, (int64_t)sms * 2);
        k_nn_mma<<<nbt, 128, smem_t, s>>>(N, h->model.n_types, h->model.n_neurons, HP, h->nn_stride, h->d_nn, h->b1U, h->b1q, h->d_xyzt,
                                          h->d_D, h->d_Ui, h->d_qraw, h->d_FpU, h->d_FpQ, h->d_sums);
    } else if (h->ND == QNEP_NDESC) {
        k_nn<<<nb, NN_BLOCK, smem, s>>>(N, h->model.n_types, h->model.n_neurons, h->nn_stride, h->d_nn, h->b1U, h->b1q, h->d_xyzt,
                                        h->d_D, h->d_Ui, h->d_qraw, h->d_FpU, h->d_FpQ, h->d_sums);
    } else {
        static bool attr1 = false;
        if (!attr1) { QNEP_CUDA_OK(h, cudaFuncSetAttribute(k_nn1<QNEP_NDESC_HB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)); attr1 = true; }
        const int nb1 = (int)std::min<int64_t>((N + 127) / 128, (int64_t)sms * 3);
        k_nn1<QNEP_NDESC_HB><<<nb1, 128, smem, s>>>(N, h->model.n_types, h->model.n_neurons, h->nn_stride, h->d_nn, h->b1U, h->b1q, h->d_xyzt,
                                                    h->d_D, h->d_Ui, h->d_qraw, h->d_FpU, h->d_FpQ, h->d_sums);
    }
    const int nb2 = (int)((N + 255) / 256);
    k_neutralise<<<nb2, 256, 0, s>>>(N, h->d_qraw, h->d_sums, h->model.q_total, h->d_sidx, h->d_cm, h->d_q, h->d_qcm, charges_out);
    h->launches += 2;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int qnep_launch_force_angular(qnep_handle* h, bool bec, bool virial, bool atomv, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + ANG_BLOCK - 1) / ANG_BLOCK);
    const float rcinv = (float)(1.0 / h->model.rc_a);
    QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_Facc, 0, sizeof(float) * (bec ? 9 : (atomv ? 12 : 3)) * N, s));
    dispatch_T(h->model.n_types, [&](auto t) {
        constexpr int T = decltype(t)::value;
#define QNEP_FA(B, V, A, Z) k_force_angular<T, B, V, A, Z><<<nb, ANG_BLOCK, 0, s>>>(N, h->d_xyzt, h->d_lvA, h->capLA, h->d_nlvA, h->d_cA, h->d_cR, rcinv, \
                                                                                     h->d_FpU, h->d_FpQ, h->d_phi, (float)h->model.sqrt_eps_inf, \
                                                                                     h->d_A, h->d_Fp, h->d_recA, h->d_recB, h->d_Facc, h->d_sums, h->zbl, h->ND == QNEP_NDESC_HB ? 1 : 0)
        const bool zb = h->zbl.on != 0;
        if (bec) QNEP_FA(true, false, false, false);                 // the Born effective charges do not see the ZBL core
        else if (atomv) { if (zb) QNEP_FA(false, true, true, true); else QNEP_FA(false, true, true, false); }
        else if (virial) { if (zb) QNEP_FA(false, true, false, true); else QNEP_FA(false, true, false, false); }
        else { if (zb) QNEP_FA(false, false, false, true); else QNEP_FA(false, false, false, false); }
#undef QNEP_FA
    });
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

// must follow qnep_launch_force_angular of the same mode (it writes the gather records and the angular accumulator)
int qnep_launch_force_radial(qnep_handle* h, bool bec, bool virial, double* out, double* atomv_out, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + RAD_BLOCK - 1) / RAD_BLOCK);
    const float rcinv = (float)(1.0 / h->model.rc_r);
    dispatch_T(h->model.n_types, [&](auto t) {
        constexpr int T = decltype(t)::value;
#define QNEP_FR(B, V) k_force_radial<T, B, V><<<nb, RAD_BLOCK, 0, s>>>(N, h->geo, h->d_recA, h->d_recB, h->d_xyzt, h->d_lvR, h->capLR, h->d_nlvR, \
                                                                        h->d_lvRend, rcinv, h->d_Facc, h->d_Fs, h->d_q,                  \
                                                                        (float)h->model.sqrt_eps_inf, h->d_sidx, out, h->d_sums, nullptr, nullptr)
        if (bec) QNEP_FR(true, false);
        else if (atomv_out) k_force_radial<T, false, true, true><<<nb, RAD_BLOCK, 0, s>>>(N, h->geo, h->d_recA, h->d_recB, h->d_xyzt, h->d_lvR, h->capLR, h->d_nlvR,
                                                                                          h->d_lvRend, rcinv, h->d_Facc, h->d_Fs, h->d_q, (float)h->model.sqrt_eps_inf,
                                                                                          h->d_sidx, out, h->d_sums, h->d_Wat, atomv_out);
        else if (virial) QNEP_FR(false, true);
        else QNEP_FR(false, false);
#undef QNEP_FR
    });
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

// FP32 FMA throughput of this device (TFLOP/s), timed with CUDA events on `s`
int qnep_launch_fma_peak(double* tflops_host, cudaStream_t s)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return QNEP_ERR_CUDA;
    float* d = nullptr;
    if (cudaMalloc(&d, sizeof(float)) != cudaSuccess) return QNEP_ERR_OOM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms * 8, iters = 4096;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, s);
        k_fma_peak<<<blocks, 256, 0, s>>>(iters, 1.f + rep, d);
        cudaEventRecord(e1, s);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return QNEP_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 16.0 * iters * 256.0 * blocks;
        if (rep > 0 && ms > 0.f) best = std::max(best, flops / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d);
    *tflops_host = best;
    return QNEP_OK;
}
