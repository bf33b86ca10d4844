// qnep_internal.cuh -- handle layout and launcher prototypes shared by the .cu files of the
// B200-native qNEP force evaluation (arXiv 2601.19034).  Not part of the public boundary
// (include/qnep.h).  Shares nothing with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/qnep.h"

#define QNEP_MAX_TYPES 4
#define QNEP_NLM 24                 // real harmonics l = 1..4: 3 + 5 + 7 + 9
#define QNEP_NL_MASK 0x03ffffff     // neighbour entry: low 26 bits = sorted atom index, high 6 bits = cell offset of the image
#define QNEP_NL_SHIFT 26            // (three signed 2-bit fields d0, d1, d2 in {-1, 0, 1}, d0 in the top bits); pair lists: species
#define QNEP_KPAD 12                // Chebyshev coefficient rows padded from 9 to 12 floats (3 x float4)
#define QNEP_NB 9                   // basis functions k = 0..8 (basis_r = basis_a = 8 in this version)
#define QNEP_NRAD 5                 // n = 0..4
#define QNEP_NDESC 25               // radial + 3-body angular descriptors
#define QNEP_NDESC_HB 35            // with NEP4's 4- and 5-body terms (rows 25..29 and 30..34)
#define QNEP_GRAPH_MAX_ATOMS 100000   // above this the step is not launch-bound and keeps its per-stage events
// PPPM mesh bins of the sweep kernel (pppm_sweep.cu): bin edge in mesh points along x, y, z
#define QNEP_MB_X 4
#define QNEP_MB_Y 8
#define QNEP_MB_Z 8
#define QNEP_SWEEP_MIN_ATOMS 20000    // below this the per-atom spread kernel is used (too few columns to fill the GPU)

// Neighbour lists are WARP-TILED: the rows of the 32 atoms p = 32 w .. 32 w + 31 are interleaved in one contiguous
// block, so a warp streams its lists sequentially (one DRAM page after the other) and every thread loads 16 bytes
// per request.  Packed-word lists (skin list, live radial list) keep four consecutive slots of an atom in one int4:
//     vector (g, p) at  ((p >> 5) * (cap / 4) + g) * 32 + (p & 31)          [int4 units], slots 4g .. 4g+3
// and the live angular pairs one float4 per slot:
//     entry (s, p)  at  ((p >> 5) * cap + s) * 32 + (p & 31)                [float4 units].
// Slots at and beyond an atom's count are undefined: readers never look at them.
#define QNEP_TILE 32
#define QNEP_NL_EMPTY (-1)           // filler of the last int4 of a live list (never read: readers stop at the count)
__host__ __device__ __forceinline__ int64_t qnep_tiled_base(int64_t p, int rows_per_atom)
{
    return ((p >> 5) * (int64_t)rows_per_atom) * QNEP_TILE + (p & 31);
}

// The cell offset is decoded with shifts and added with one FMA per component (a table in shared memory cost 4-5 L1
// wavefronts per neighbour in kernels that are bound by L1 wavefronts):  d += (d0, d1, d2) * (h0, h1, h2).
__host__ __device__ __forceinline__ int qnep_image_bits(int d0, int d1, int d2)
{
    return (int)(((unsigned)(d0 & 3) << 30) | ((unsigned)(d1 & 3) << 28) | ((unsigned)(d2 & 3) << 26));
}
struct CellVecs { float c[9]; int tri; };      // Geometry::cellv in registers
__device__ __forceinline__ void qnep_add_image_shift(int e, const CellVecs& cv, float& dx, float& dy, float& dz)
{
    const float f0 = (float)(e >> 30), f1 = (float)((int)((unsigned)e << 2) >> 30), f2 = (float)((int)((unsigned)e << 4) >> 30);
    dx = fmaf(f0, cv.c[0], dx);
    dy = fmaf(f1, cv.c[4], dy);
    dz = fmaf(f2, cv.c[8], dz);
    if (cv.tri) {                                  // warp-uniform: off-diagonal parts of a non-orthogonal cell
        dx = fmaf(f1, cv.c[3], fmaf(f2, cv.c[6], dx));
        dy = fmaf(f0, cv.c[1], fmaf(f2, cv.c[7], dy));
        dz = fmaf(f0, cv.c[2], fmaf(f1, cv.c[5], dz));
    }
}
__device__ __forceinline__ CellVecs qnep_cell_vecs(const float (&cellv)[9], int tri)
{
    CellVecs cv;
#pragma unroll
    for (int k = 0; k < 9; ++k) cv.c[k] = cellv[k];
    cv.tri = tri;
    return cv;
}

constexpr double QNEP_K_COULOMB = 14.3996454784;   // eV A / e^2 (reading S9)

// device-side double accumulators
enum { SUM_E_NEP = 0, SUM_Q, SUM_PHI, SUM_U_R, SUM_U_K, SUM_U_S, SUM_W0 /* 9 entries */, SUM_KE = 15, SUM_COUNT = 16 };
// The force kernels add one 3 x 3 partial virial per BLOCK: 16 000 blocks on nine addresses serialise in L2, so they
// are spread over QNEP_WSTRIPES copies behind the named slots (stripe = block index mod QNEP_WSTRIPES); k_finalize adds
// the stripes to SUM_W0.
#define QNEP_WSTRIPES 64
#define QNEP_WSTRIDE 10              // per stripe: nine virial components, then the ZBL energy (one add per warp of k_desc_angular)
#define QNEP_SUM_ALLOC (SUM_COUNT + QNEP_WSTRIPES * QNEP_WSTRIDE)
__device__ __forceinline__ double qnep_striped_sum(const double* sums, int slot)
{
    double v = 0.0;
    for (int st = 0; st < QNEP_WSTRIPES; ++st) v += sums[SUM_COUNT + st * QNEP_WSTRIDE + slot];
    return v;
}

// Optional ZBL core (include/qnep.h qnep_set_zbl; reading Z1), passed to the angular kernels by value:
//   U(r) = kzz / r * phi(r * ainv) * f_sw(r),  phi = sum_k c_k exp(-d_k x),  f_sw the cosine switch r1 .. r2
struct ZblParams {
    int on;
    float r1, r2, r2sq, sw;              // sw = pi / (r2 - r1)
    float kzz[QNEP_MAX_TYPES][QNEP_MAX_TYPES];   // K Z_i Z_j
    float ainv[QNEP_MAX_TYPES][QNEP_MAX_TYPES];  // (Z_i^0.23 + Z_j^0.23) / 0.46850
};
__device__ __forceinline__ void qnep_zbl_eval(const ZblParams& z, int ti, int tj, float r, float rinv, float& u, float& du)
{
    const float a = z.ainv[ti][tj], x = r * a;
    const float e0 = 0.18175f * __expf(-3.19980f * x), e1 = 0.50986f * __expf(-0.94229f * x);
    const float e2 = 0.28022f * __expf(-0.40290f * x), e3 = 0.02817f * __expf(-0.20162f * x);
    const float phi = (e0 + e1) + (e2 + e3);
    const float dphi = -a * (3.19980f * e0 + 0.94229f * e1 + 0.40290f * e2 + 0.20162f * e3);
    float fsw = 1.f, dfsw = 0.f;
    if (r >= z.r1) {
        float sn, cs;
        __sincosf(z.sw * (r - z.r1), &sn, &cs);
        fsw = 0.5f + 0.5f * cs;
        dfsw = -0.5f * z.sw * sn;
    }
    const float c = z.kzz[ti][tj] * rinv;
    u = c * phi * fsw;
    du = c * (fsw * (dphi - phi * rinv) + phi * dfsw);
}
// device-side int flags
// overflow flags hold the largest count seen when a list exceeded its capacity (0 otherwise)
enum { FLAG_MAX_NR = 0 /* skin list */, FLAG_MAX_LR /* live radial */, FLAG_MAX_LA /* live angular */, FLAG_SKIN, FLAG_BAD_TYPE /* a species index outside 0..T-1 */, FLAG_TENSOR_TIMEOUT /* k_nn_umma: an MMA never completed */, FLAG_COUNT = 8 };

struct Geometry {            // periodic cell (rows of h = cell vectors a, b, c; any non-degenerate cell) and the cell grid of the neighbour search
    double L[3];             // lengths of the cell vectors (orthorhombic: the box edges)
    double hcell[3];         // |cell vector| / ncell; the search cells are h_a / ncell_a with perpendicular widths >= rc_r + skin
    double h[9];             // cell vectors, row a = h[3a .. 3a+2]
    double hinv[9];          // fractional coordinate f_b = sum_a r_a hinv[3a + b]; reciprocal vector b = 2 pi hinv[. + b]
    float cellv[9];          // edge vectors of a search cell, row a = h_a / ncell_a: the image shift of a neighbour word is d . cellv
    int triclinic;           // 0: h is diagonal (cellv too: three FMAs per shift instead of nine)
    int ncell[3];
    int ncells;
    float rc_r2, rc_a2;      // cutoffs squared
    float rcs_r2, rcs_a2;    // (cutoff + skin)^2, used at build time
    float skin_half2;        // (skin/2)^2
    // PPPM
    int grid[3];
    double hmesh_inv[3];     // N / L
};

struct qnep_handle {
    qnep_model_desc model;
    qnep_es_desc es;
    double alpha;            // resolved alpha
    std::string err;
    int64_t launches = 0;

    // model on device
    float* d_params = nullptr;       // raw copy
    float* d_cR = nullptr;           // [T*T][5][KPAD]
    float* d_cA = nullptr;           // [T*T][5][KPAD]
    float* d_nn = nullptr;           // per type: w0[H][28] (scaler folded in? no: raw), b0[H], w1U[H], w1q[H]
    int nn_stride = 0;               // floats per type in d_nn
    int nn_tensor = 0;               // qnep_set_nn_kernel: 0 packed FP32 kernel, 1 = k_nn_mma (mma.sync 3xTF32), 2 = k_nn_umma (tcgen05 3xTF32)
    int ND = QNEP_NDESC;             // descriptors per atom: 25, or 35 with the 4-/5-body terms
    int w0p = 28;                    // padded row length of w0 in d_nn (ND rounded up to a multiple of 4)
    float b1U = 0.f, b1q = 0.f;
    std::vector<float> h_params;

    // policy
    double skin = 0.0;
    int rebuild_every = 0;
    int calls_since_build = -1;      // -1: never built
    int user_capR = 0, user_capLR = 0, user_capA = 0;   // explicit capacities (qnep_set_neighbor_capacity): skin list, live radial, live angular (0: automatic)
    int grown_capR = 0, grown_capLR = 0, grown_capA = 0;   // lower bounds learnt from an overflow; the automatic estimate still applies on top
    bool force_rebuild = true;

    // workspace (sorted atom order p unless noted)
    int64_t N = 0;                   // atoms the workspace is sized for
    int capR = 0;                    // skin-list capacity (entries per atom)
    int capLR = 0, capLA = 0;        // live-list capacities
    Geometry geo;
    double box[9];
    int nkeys = 0;
    int* d_key = nullptr;            // [N] original order
    int* d_cnt = nullptr;            // [nkeys + 1]
    int* d_start = nullptr;          // [nkeys + 1]
    int* d_fill = nullptr;           // [nkeys]
    int* d_scantmp = nullptr;        // chunk totals and their scan of the multi-block exclusive scan
    size_t scantmp_len = 0;
    int* d_tmpidx = nullptr;         // [N]
    int* d_sidx = nullptr;           // [N] sorted -> original
    int* d_ctot = nullptr;           // [ncells + 1] atoms per cell (all species)
    int* d_cstart = nullptr;         // [ncells + 1] its exclusive scan
    int* d_cm = nullptr;             // [N] sorted index p -> rank q in the order of the PPPM kernels (mesh-bin order; cell-major without PPPM)
    int* d_cmi = nullptr;            // [N] q -> p
    int nmb[3] = {0, 0, 0};          // PPPM mesh bins per axis (grid / QNEP_MB_*); nmbins = 0 when PPPM is off
    int nmbins = 0;
    int* d_mbkey = nullptr;          // [N] mesh-bin key of sorted atom p (build time)
    int* d_mbcnt = nullptr;          // [nmbins + 1]
    int* d_mbstart = nullptr;        // [nmbins + 1] first mesh-bin-order rank q of every bin
    int* d_mbfill = nullptr;         // [nmbins]
    int pppm_kernels = 0;            // 0 automatic, 1 per-atom spread / gather, 2 sweep kernels (qnep_set_pppm_kernels)
    int2* d_qcm = nullptr;           // [N] mesh-bin order: (sorted index p, bits of the neutralised charge q_p) for the PPPM sweep kernels
    alignas(64) CUtensorMap tm_mesh;  // TMA descriptor of the charge mesh (box 4 x 14 x 16 floats) for k_spread_sweep; valid when tm_ok
    bool tm_ok = false;
    int* d_cellc = nullptr;          // [N] packed cell coordinates (10 bits each)
    float4* d_xyzt = nullptr;        // [N] cell-relative position, w = type bits
    float4* d_off0 = nullptr;        // [N] the same at build time (skin check)
    float4* d_mfrac = nullptr;       // [N] PPPM: fractional mesh offsets (dx, dy, dz, bits of the packed nearest mesh point), mesh-bin order
    int* d_mi0 = nullptr;            // [N] PPPM: nearest mesh point, packed 10 bits each, cell-major order
    int4* d_nlR = nullptr;           // warp-tiled [capR / 4] int4 per atom: skin list (r < rc_r + skin at build time)
    int* d_nnR = nullptr;            // [N] slots of the skin list (every species segment padded to a multiple of 4)
    int* d_nnR0 = nullptr;           // [N] neighbours in the skin list (statistics)
    int* d_nlRend = nullptr;         // [T][N] end slot of the species-t segment of the skin list
    int4* d_lvR = nullptr;           // warp-tiled [capLR / 4] int4 per atom: live radial list of this step (r < rc_r)
    int* d_nlvR = nullptr;           // [N]
    int* d_lvRend = nullptr;         // [T][N] end of the species-t segment of the (type-major) live radial list
    float4* d_lvA = nullptr;         // warp-tiled [capLA] float4 per atom: live angular pairs (dx, dy, dz, bits(j | tj << 26))
    int* d_nlvA = nullptr;           // [N]
    float* d_D = nullptr;            // [25][N]
    float* d_A = nullptr;            // [5*24][N]
    float* d_Ui = nullptr;           // [N]
    float* d_qraw = nullptr;         // [N]
    float* d_q = nullptr;            // [N]
    float* d_FpU = nullptr;          // [25][N]
    float* d_FpQ = nullptr;          // [25][N]
    float* d_Fp = nullptr;           // [25][N]
    float* d_recA = nullptr;         // [T][N][8] gather records of the radial force kernel: (x, y, z, P^t_0..P^t_4)
    float4* d_recB = nullptr;        // [T][N]    (P^t_5..P^t_8),  P^t_k = sum_n Fp_n c^{ti t}_{nk}
    float* d_phik = nullptr;         // [N]
    float* d_phir = nullptr;         // [N]
    float* d_phi = nullptr;          // [N]
    float* d_Fs = nullptr;           // [3][N] static electrostatic force
    float* d_Facc = nullptr;         // [12][N] fp32 accumulators of the angular pass (atomics): rows 0-2 force (rows 0-8 Z in BEC
                                     // mode), rows 3-11 per-atom virial (qnep_compute_atom_virial)
    float* d_Wat = nullptr;          // [9][N] per-atom virial, static electrostatic parts (allocated on first use)
    double* d_sums = nullptr;        // [SUM_COUNT]
    int* d_flags = nullptr;          // [FLAG_COUNT]
    int* h_flags = nullptr;          // pinned
    cudaEvent_t ev_flags = nullptr;
    bool flags_pending = false;
    double* d_Fmd = nullptr;         // [3][N] forces kept for qnep_md_run (original order)
    bool md_have_forces = false;
    uint32_t md_want = 0;            // extra outputs of the evaluations inside qnep_md_run (qnep_md_set_outputs)
    double* md_virial = nullptr;
    double* md_charges = nullptr;
    ZblParams zbl = {};              // optional ZBL core (qnep_set_zbl)

    // Ewald
    int nk = 0;
    float4* d_kvec = nullptr;        // [nk] (kx, ky, kz, G)
    int* d_kint = nullptr;           // [nk] packed integers
    int ew_nmax = 0;
    float2* d_ephase = nullptr;      // [3][nmax+1][N]
    double2* d_S = nullptr;          // [nk]
    // PPPM
    int64_t ngrid = 0;
    int64_t nhalf = 0;               // elements of d_half
    float* d_mesh = nullptr;         // [Nx][Ny][Nz] real charge mesh
    float2* d_half = nullptr;        // half-spectrum array of the forward transform [x][y][N2/2 + 16] (N2 >= 32)
    float2* d_cm1 = nullptr;         // complex meshes
    float2* d_cm2 = nullptr;
    float2* d_cm3 = nullptr;         // third complex mesh: per-atom virial pass only (allocated on first use)
    int64_t cm3_ngrid = 0;           // mesh points d_cm3 was allocated for (checked against ngrid before every use)
    float4* d_field = nullptr;       // [Nx][Ny][Nz] (Phi, E_x, E_y, E_z)
    float* d_gtab = nullptr;         // 1-D influence tables: per axis N entries of (A_alpha) then k_alpha
    float2* d_twiddle = nullptr;     // per axis twiddles
    int tw_n = 0;

    // qnep_md_run: one CUDA graph per step kind (0: lists reused, 1: rebuild), replayed while the key is unchanged
    int md_graph_mode = 1;                 // 0 never, 1 when N <= QNEP_GRAPH_MAX_ATOMS (launch-bound sizes), 2 always
    cudaGraphExec_t md_exec[2] = {nullptr, nullptr};
    int64_t md_exec_launches[2] = {0, 0};
    struct MdKey { const void *pos, *vel, *types, *virial, *charges; int64_t N; double dt; double m[QNEP_MAX_TYPES]; cudaStream_t s; uint64_t gen; uint64_t want; } md_key = {};
    cudaStream_t md_stream = nullptr;      // graphs run on an own stream (the legacy default stream cannot be captured), fenced by events
    cudaEvent_t md_fence = nullptr;
    uint64_t ws_generation = 0;            // bumped whenever workspace pointers, capacities or the geometry change

    // host staging (qnep_compute_host); the charges go back on a second stream while the PPPM and force kernels run
    cudaStream_t copy_stream = nullptr; cudaEvent_t ev_q_ready = nullptr, ev_q_copied = nullptr;
    double* early_q_host = nullptr; const double* early_q_dev = nullptr;
    double* d_hpos = nullptr; int32_t* d_htypes = nullptr; double* d_hout = nullptr; int64_t hostN = 0;

    // timing
    static constexpr int NEV = QNEP_T_COUNT;   // events per evaluation: QNEP_T_TOTAL stage boundaries + 1
    static constexpr int RING = 512;           // evaluations kept for qnep_profile_sum
    std::vector<cudaEvent_t> ring;             // [RING][NEV]
    int64_t prof_count = 0;                    // evaluations since qnep_profile_reset
    cudaEvent_t* ev = nullptr;                 // event set of the last evaluation
    bool ev_valid = false;
    bool rebuilt_last = false;
    cudaStream_t last_stream = nullptr;
};

#define QNEP_CUDA_OK(h, call)                                                              \
    do {                                                                                   \
        cudaError_t e__ = (call);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            (h)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                \
            return e__ == cudaErrorMemoryAllocation ? QNEP_ERR_OOM : QNEP_ERR_CUDA;        \
        }                                                                                  \
    } while (0)

// ---- launchers (each enqueues kernels on `s` and bumps h->launches) ----
// neighbor.cu
int qnep_launch_build(qnep_handle* h, const double* pos, const int32_t* types, cudaStream_t s);
int qnep_launch_prep(qnep_handle* h, const double* pos, bool at_build, cudaStream_t s);
int qnep_launch_list_stats(qnep_handle* h, double out[6], cudaStream_t s);
// descriptor.cu
int qnep_launch_pairs(qnep_handle* h, cudaStream_t s);
int qnep_launch_desc_angular(qnep_handle* h, cudaStream_t s);       // adds the ZBL energy when the core is on
int qnep_launch_nn(qnep_handle* h, double* charges_out, cudaStream_t s);
int qnep_launch_force_angular(qnep_handle* h, bool bec, bool virial, bool atomv, cudaStream_t s);
int qnep_launch_force_radial(qnep_handle* h, bool bec, bool virial, double* out, double* atomv_out, cudaStream_t s);
int qnep_launch_fma_peak(double* tflops_host, cudaStream_t s);
// electro.cu
int qnep_launch_realspace(qnep_handle* h, bool atomv, cudaStream_t s);
int qnep_launch_phi_finalize(qnep_handle* h, cudaStream_t s);
int qnep_setup_ewald(qnep_handle* h);
int qnep_launch_ewald(qnep_handle* h, const double* pos, bool atomv, cudaStream_t s);
// pppm.cu
int qnep_setup_pppm(qnep_handle* h);
int qnep_launch_pppm(qnep_handle* h, bool virial, cudaStream_t s);
int qnep_launch_pppm_atom_virial(qnep_handle* h, cudaStream_t s);
// pppm_sweep.cu
bool qnep_sweep_usable(const qnep_handle* h);
int qnep_setup_sweep(qnep_handle* h);
int qnep_launch_spread_sweep(qnep_handle* h, cudaStream_t s);
