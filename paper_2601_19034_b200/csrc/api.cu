// api.cu -- the C ABI of include/qnep.h: handle management and the per-step pipeline
// (SURVEY.md 8(a) steps a1-a12 in order).  Host code only orchestrates; every step runs in the
// CUDA kernels of neighbor.cu, descriptor.cu, electro.cu and pppm.cu.
#include "qnep_internal.cuh"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>

namespace {

std::string g_create_error;

template <typename Tp>
int dev_alloc(qnep_handle* h, Tp** p, size_t count)
{
    if (*p) { cudaFree(*p); *p = nullptr; }
    QNEP_CUDA_OK(h, cudaMalloc((void**)p, sizeof(Tp) * std::max<size_t>(count, 1)));
    return QNEP_OK;
}

void free_workspace(qnep_handle* h)
{
    void** ptrs[] = {(void**)&h->d_key, (void**)&h->d_cnt, (void**)&h->d_start, (void**)&h->d_fill, (void**)&h->d_tmpidx,
                     (void**)&h->d_sidx, (void**)&h->d_cm, (void**)&h->d_cmi, (void**)&h->d_cellc, (void**)&h->d_xyzt, (void**)&h->d_off0, (void**)&h->d_mfrac,
                     (void**)&h->d_mi0, (void**)&h->d_nlR, (void**)&h->d_nnR, (void**)&h->d_nnR0, (void**)&h->d_nlRend, (void**)&h->d_lvR, (void**)&h->d_nlvR,
                     (void**)&h->d_lvA, (void**)&h->d_nlvA, (void**)&h->d_D, (void**)&h->d_A, (void**)&h->d_Ui, (void**)&h->d_qraw,
                     (void**)&h->d_q, (void**)&h->d_FpU, (void**)&h->d_FpQ, (void**)&h->d_Fp, (void**)&h->d_recA, (void**)&h->d_recB, (void**)&h->d_lvRend,
                     (void**)&h->d_phik, (void**)&h->d_phir, (void**)&h->d_phi, (void**)&h->d_Fs, (void**)&h->d_Facc,
                     (void**)&h->d_Fmd, (void**)&h->d_mbkey, (void**)&h->d_qcm};
    for (void** p : ptrs) { if (*p) cudaFree(*p); *p = nullptr; }
    h->N = 0;
    h->md_have_forces = false;
}

int validate_es(qnep_handle* h, const qnep_es_desc* es)
{
    if (es->method < 0 || es->method > 2) { h->err = "es.method must be 0, 1 or 2"; return QNEP_ERR_INVALID_ARG; }
    if (es->method == 2) {
        if (es->order != 5) { h->err = "PPPM order must be 5"; return QNEP_ERR_UNSUPPORTED; }
        for (int a = 0; a < 3; ++a) {
            const int n = es->grid[a];
            if (n < 16 || n > 512 || (n & (n - 1))) { h->err = "PPPM grid must be a power of two in 16..512"; return QNEP_ERR_UNSUPPORTED; }
        }
    }
    return QNEP_OK;
}

// geometry for a box (rows = cell vectors, any non-degenerate cell); returns UNSUPPORTED for boxes narrower than r_c + skin
int make_geometry(qnep_handle* h, const double box[9], Geometry* g)
{
    const double rcs = h->model.rc_r + h->skin;
    const double* B = box;
    const double det = B[0] * (B[4] * B[8] - B[5] * B[7]) - B[1] * (B[3] * B[8] - B[5] * B[6]) + B[2] * (B[3] * B[7] - B[4] * B[6]);
    if (!(std::fabs(det) > 1e-12)) { h->err = "degenerate box (zero volume)"; return QNEP_ERR_INVALID_ARG; }
    // inverse (adjugate / det): hinv[3a + b] = (h^-1)_{ab}
    g->hinv[0] = (B[4] * B[8] - B[5] * B[7]) / det; g->hinv[1] = (B[2] * B[7] - B[1] * B[8]) / det; g->hinv[2] = (B[1] * B[5] - B[2] * B[4]) / det;
    g->hinv[3] = (B[5] * B[6] - B[3] * B[8]) / det; g->hinv[4] = (B[0] * B[8] - B[2] * B[6]) / det; g->hinv[5] = (B[2] * B[3] - B[0] * B[5]) / det;
    g->hinv[6] = (B[3] * B[7] - B[4] * B[6]) / det; g->hinv[7] = (B[1] * B[6] - B[0] * B[7]) / det; g->hinv[8] = (B[0] * B[4] - B[1] * B[3]) / det;
    g->triclinic = (box[1] != 0 || box[2] != 0 || box[3] != 0 || box[5] != 0 || box[6] != 0 || box[7] != 0) ? 1 : 0;
    g->ncells = 1;
    for (int a = 0; a < 3; ++a) {
        for (int c = 0; c < 3; ++c) g->h[3 * a + c] = box[3 * a + c];
        g->L[a] = std::sqrt(box[3 * a] * box[3 * a] + box[3 * a + 1] * box[3 * a + 1] + box[3 * a + 2] * box[3 * a + 2]);
        if (!(g->L[a] > 0)) { h->err = "box edge must be positive"; return QNEP_ERR_INVALID_ARG; }
        // perpendicular width of the cell along a: 1 / |reciprocal vector a| (= L_a for an orthorhombic box)
        const double width = 1.0 / std::sqrt(g->hinv[a] * g->hinv[a] + g->hinv[3 + a] * g->hinv[3 + a] + g->hinv[6 + a] * g->hinv[6 + a]);
        if (width < rcs) { h->err = "box narrower than r_c + skin"; return QNEP_ERR_UNSUPPORTED; }
        g->ncell[a] = std::min(1023, std::max(1, (int)floor(width / rcs)));
        g->hcell[a] = g->L[a] / g->ncell[a];
        for (int c = 0; c < 3; ++c) g->cellv[3 * a + c] = (float)(box[3 * a + c] / g->ncell[a]);
        g->ncells *= g->ncell[a];
        g->grid[a] = h->es.method == 2 ? h->es.grid[a] : 0;
        g->hmesh_inv[a] = g->grid[a] > 0 ? g->grid[a] / g->L[a] : 0.0;
    }
    g->rc_r2 = (float)(h->model.rc_r * h->model.rc_r);
    g->rc_a2 = (float)(h->model.rc_a * h->model.rc_a);
    g->rcs_r2 = (float)(rcs * rcs);
    g->rcs_a2 = (float)((h->model.rc_a + h->skin) * (h->model.rc_a + h->skin));
    g->skin_half2 = (float)(0.25 * h->skin * h->skin);
    return QNEP_OK;
}

int ensure_workspace(qnep_handle* h, int64_t N, const double box[9])
{
    Geometry g;
    int rc = make_geometry(h, box, &g);
    if (rc) return rc;
    const bool box_changed = std::memcmp(box, h->box, sizeof(double) * 9) != 0;
    const double vol = std::fabs(g.h[0] * (g.h[4] * g.h[8] - g.h[5] * g.h[7]) - g.h[1] * (g.h[3] * g.h[8] - g.h[5] * g.h[6]) +
                                 g.h[2] * (g.h[3] * g.h[7] - g.h[4] * g.h[6]));
    const double rho = (double)N / vol;
    auto cap_for = [&](double rc_, int user, int grown) {
        if (user > 0) return (user + 3) / 4 * 4;          // packed-word lists hold four slots per int4
        const double expect = 4.0 / 3.0 * M_PI * rc_ * rc_ * rc_ * rho;
        return std::max(((int)(expect * 1.5) + 24 + 3) / 4 * 4, grown);
    };
    const int capR = cap_for(h->model.rc_r + h->skin, h->user_capR, h->grown_capR);     // skin list
    const int capLR = cap_for(h->model.rc_r, h->user_capLR, h->grown_capLR);            // live radial list
    const int capLA = cap_for(h->model.rc_a, h->user_capA, h->grown_capA);              // live angular pairs
    const int T = h->model.n_types;
    const int nkeys = T * g.ncells;
    const bool realloc_atoms = N != h->N || capR != h->capR || capLR != h->capLR || capLA != h->capLA;
    if (realloc_atoms) {
        free_workspace(h);
        const size_t n = (size_t)N;
        if ((rc = dev_alloc(h, &h->d_key, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_tmpidx, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_sidx, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_cm, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_cmi, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_mbkey, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_qcm, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_cellc, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_xyzt, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_off0, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_mfrac, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_mi0, n))) return rc;
        const size_t npad = (n + QNEP_TILE - 1) / QNEP_TILE * QNEP_TILE;
        if ((rc = dev_alloc(h, &h->d_nlR, npad * (capR / 4)))) return rc;
        if ((rc = dev_alloc(h, &h->d_nnR, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_nnR0, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_nlRend, n * T))) return rc;
        if ((rc = dev_alloc(h, &h->d_lvR, npad * (capLR / 4)))) return rc;
        if ((rc = dev_alloc(h, &h->d_nlvR, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_lvA, npad * capLA))) return rc;
        if ((rc = dev_alloc(h, &h->d_nlvA, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_D, n * h->ND))) return rc;
        if ((rc = dev_alloc(h, &h->d_A, n * QNEP_NRAD * QNEP_NLM))) return rc;
        if ((rc = dev_alloc(h, &h->d_Ui, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_qraw, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_q, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_FpU, n * h->ND))) return rc;
        if ((rc = dev_alloc(h, &h->d_FpQ, n * h->ND))) return rc;
        if ((rc = dev_alloc(h, &h->d_Fp, n * h->ND))) return rc;
        if ((rc = dev_alloc(h, &h->d_recA, n * T * 8))) return rc;
        if ((rc = dev_alloc(h, &h->d_recB, n * T))) return rc;
        if ((rc = dev_alloc(h, &h->d_lvRend, n * T))) return rc;
        if ((rc = dev_alloc(h, &h->d_phik, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_phir, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_phi, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_Fs, n * 3))) return rc;
        if ((rc = dev_alloc(h, &h->d_Facc, n * 12))) return rc;
        if (h->d_Wat) { cudaFree(h->d_Wat); h->d_Wat = nullptr; }
        if ((rc = dev_alloc(h, &h->d_Fmd, n * 3))) return rc;
        h->N = N; h->capR = capR; h->capLR = capLR; h->capLA = capLA;
        QNEP_CUDA_OK(h, cudaMemset(h->d_nlvR, 0, sizeof(int) * n));
        QNEP_CUDA_OK(h, cudaMemset(h->d_nlvA, 0, sizeof(int) * n));
        h->force_rebuild = true;
    }
    if (nkeys != h->nkeys || !h->d_cnt) {
        if ((rc = dev_alloc(h, &h->d_cnt, (size_t)nkeys + 1))) return rc;
        if ((rc = dev_alloc(h, &h->d_start, (size_t)nkeys + 1))) return rc;
        if ((rc = dev_alloc(h, &h->d_fill, (size_t)nkeys))) return rc;
        if ((rc = dev_alloc(h, &h->d_ctot, (size_t)g.ncells + 1))) return rc;
        if ((rc = dev_alloc(h, &h->d_cstart, (size_t)g.ncells + 1))) return rc;
        h->nkeys = nkeys;
        h->ws_generation += 1;
        h->force_rebuild = true;
    }
    {
        // PPPM mesh bins (pppm_sweep.cu, k_mbin_key)
        int nmb[3] = {0, 0, 0}, nmbins = 0;
        if (h->es.method == 2) {
            nmb[0] = g.grid[0] / QNEP_MB_X; nmb[1] = g.grid[1] / QNEP_MB_Y; nmb[2] = g.grid[2] / QNEP_MB_Z;
            nmbins = nmb[0] * nmb[1] * nmb[2];
        }
        if (nmbins != h->nmbins || (nmbins > 0 && !h->d_mbcnt)) {
            if ((rc = dev_alloc(h, &h->d_mbcnt, (size_t)nmbins + 1))) return rc;
            if ((rc = dev_alloc(h, &h->d_mbstart, (size_t)nmbins + 1))) return rc;
            if ((rc = dev_alloc(h, &h->d_mbfill, (size_t)nmbins + 1))) return rc;
            h->nmbins = nmbins;
            h->ws_generation += 1;
            h->force_rebuild = true;
        }
        for (int a = 0; a < 3; ++a) h->nmb[a] = nmb[a];
    }
    {
        // scratch of the multi-block scan: 2 (chunks + 1) ints for the longer of the two key arrays (2048 keys per chunk)
        const size_t need = 2 * ((size_t)std::max(nkeys, h->nmbins) / 2048 + 2);
        if (need > h->scantmp_len) {
            if ((rc = dev_alloc(h, &h->d_scantmp, need))) return rc;
            h->scantmp_len = need;
            h->ws_generation += 1;
        }
    }
    const bool geo_changed = box_changed || std::memcmp(&g, &h->geo, sizeof(Geometry)) != 0;
    h->geo = g;
    std::memcpy(h->box, box, sizeof(double) * 9);
    if (geo_changed || realloc_atoms) {
        h->ws_generation += 1;
        h->force_rebuild = true;
        // the table uploads below are synchronous copies on the legacy stream: kernels of the previous (asynchronous)
        // call on a non-blocking caller stream may still be reading the old tables
        if (h->flags_pending) QNEP_CUDA_OK(h, cudaStreamSynchronize(h->last_stream));
        if (h->es.method == 1) { if ((rc = qnep_setup_ewald(h))) return rc; }
        if (h->es.method == 2) { if ((rc = qnep_setup_pppm(h))) return rc; }
    }
    return QNEP_OK;
}

// translate the flags copied back by the previous call
int consume_flags(qnep_handle* h)
{
    h->flags_pending = false;
    const int* f = h->h_flags;
    // the device flags are sticky (a rebuild inside qnep_md_run must not erase a violation seen earlier in the
    // run): they are cleared here, on the error path only, once the host has read them
    if (f[FLAG_MAX_NR] || f[FLAG_MAX_LR] || f[FLAG_MAX_LA] || f[FLAG_SKIN] || f[FLAG_BAD_TYPE] || f[FLAG_TENSOR_TIMEOUT]) {
        cudaMemsetAsync(h->d_flags, 0, sizeof(int) * FLAG_COUNT, h->last_stream);
        cudaStreamSynchronize(h->last_stream);
    }
    if (f[FLAG_TENSOR_TIMEOUT]) {
        h->err = "k_nn_umma: a tensor-core operation did not complete";
        return QNEP_ERR_CUDA;
    }
    if (f[FLAG_BAD_TYPE]) {
        h->err = "types_dev holds a species index outside 0..n_types-1";
        h->force_rebuild = true;
        return QNEP_ERR_INVALID_ARG;
    }
    if (f[FLAG_MAX_NR] > h->capR || f[FLAG_MAX_LR] > h->capLR || f[FLAG_MAX_LA] > h->capLA) {
        h->err = "neighbour list capacity exceeded (skin list " + std::to_string(f[FLAG_MAX_NR]) + "/" + std::to_string(h->capR) +
                 ", live radial " + std::to_string(f[FLAG_MAX_LR]) + "/" + std::to_string(h->capLR) + ", live angular " +
                 std::to_string(f[FLAG_MAX_LA]) + "/" + std::to_string(h->capLA) + "); capacity grown, call again";
        auto grow = [](int cap, int seen) { return std::max(cap, (seen * 5 / 4 + 8 + 3) / 4 * 4); };
        // the grown values are lower bounds on top of the automatic estimate (a stale one can only be too generous);
        // an explicit capacity that proved too small is dropped
        if (f[FLAG_MAX_NR] > h->capR) {
            // the truncated skin list hid the true live counts: scale them from the skin-list count by the volume ratios
            h->grown_capR = grow(h->capR, f[FLAG_MAX_NR]);
            const double rcs = h->model.rc_r + h->skin;
            const double fr = std::pow(h->model.rc_r / rcs, 3.0), fa = std::pow(h->model.rc_a / rcs, 3.0);
            h->grown_capLR = grow(h->capLR, (int)(f[FLAG_MAX_NR] * fr * 1.1) + 1);
            h->grown_capA = grow(h->capLA, (int)(f[FLAG_MAX_NR] * fa * 1.3) + 1);
            h->user_capR = h->user_capLR = h->user_capA = 0;
        }
        if (f[FLAG_MAX_LR] > h->capLR) { h->grown_capLR = grow(h->capLR, f[FLAG_MAX_LR]); h->user_capLR = 0; }
        if (f[FLAG_MAX_LA] > h->capLA) { h->grown_capA = grow(h->capLA, f[FLAG_MAX_LA]); h->user_capA = 0; }
        h->force_rebuild = true;
        return QNEP_ERR_NEIGHBOR_OVERFLOW;
    }
    if (f[FLAG_SKIN]) {
        h->err = "an atom moved more than skin/2 since the last neighbour build";
        h->force_rebuild = true;
        return QNEP_ERR_SKIN_VIOLATED;
    }
    return QNEP_OK;
}

__global__ void k_finalize(const double* __restrict__ sums, int mode, double* __restrict__ energy, double* __restrict__ virial)
{
    if (threadIdx.x == 0 && energy) {
        double e = sums[SUM_E_NEP] + sums[SUM_U_K] + qnep_striped_sum(sums, 9);      // stripe slot 9: ZBL energy
        if (mode == 1) e += sums[SUM_U_R] + sums[SUM_U_S];
        energy[0] = e;
    }
    if (threadIdx.x < 9 && virial) virial[threadIdx.x] = sums[SUM_W0 + threadIdx.x] + qnep_striped_sum(sums, threadIdx.x);
}

// ---- debug / parity helpers -----------------------------------------------------------------------
__global__ void k_dbg_rows(int64_t N, int ncomp, const float* __restrict__ src, const int* __restrict__ sidx,
                           int atom_major, double* __restrict__ dst)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int64_t i = sidx[p];
    for (int v = 0; v < ncomp; ++v) {
        const double x = src[(int64_t)v * N + p];
        if (atom_major) dst[i * ncomp + v] = x; else dst[(int64_t)v * N + i] = x;
    }
}

__global__ void k_dbg_copy(int64_t n, const float* __restrict__ src, double* __restrict__ dst)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[i];
}

__global__ void k_dbg_energy(const double* __restrict__ sums, double* __restrict__ dst)
{
    dst[0] = sums[SUM_E_NEP] + qnep_striped_sum(sums, 9);      // short-ranged part: network site energies + ZBL core
    dst[1] = sums[SUM_U_R]; dst[2] = sums[SUM_U_K]; dst[3] = sums[SUM_U_S];
}

// ---- velocity-Verlet kernels ----------------------------------------------------------------------
struct Masses { double m[QNEP_MAX_TYPES]; };

__global__ void k_vv_kick_drift(int64_t N, double* __restrict__ pos, double* __restrict__ vel, const double* __restrict__ F,
                                const int32_t* __restrict__ types, Masses ms, double dt)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double im = 0.5 * dt / ms.m[types[i]];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double v = vel[a * N + i] + im * F[a * N + i];
        vel[a * N + i] = v;
        pos[a * N + i] += dt * v;
    }
}

__global__ void k_vv_kick(int64_t N, double* __restrict__ vel, const double* __restrict__ F, const int32_t* __restrict__ types,
                          Masses ms, double dt, double* __restrict__ sums)
{
    __shared__ double sh[32];
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double ke = 0.0;
    if (i < N) {
        const double m = ms.m[types[i]];
        const double im = 0.5 * dt / m;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            const double v = vel[a * N + i] + im * F[a * N + i];
            vel[a * N + i] = v;
            ke += 0.5 * m * v * v;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ke += __shfl_xor_sync(0xffffffffu, ke, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = ke;
    __syncthreads();
    if (threadIdx.x < 32) {
        double r = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xffffffffu, r, o);
        if (threadIdx.x == 0) atomicAdd(&sums[SUM_KE], r);
    }
}

__global__ void k_md_energy(const double* __restrict__ sums, int mode, double* __restrict__ out)
{
    double e = sums[SUM_E_NEP] + sums[SUM_U_K] + qnep_striped_sum(sums, 9);
    if (mode == 1) e += sums[SUM_U_R] + sums[SUM_U_S];
    out[0] = e;
    out[1] = sums[SUM_KE];
}

// ---- Eq. 29-30: external-field force and polarization current from the Born effective charges -------------
struct Vec3d { double v[3]; };

__global__ void __launch_bounds__(256)
k_response(int64_t N, const double* __restrict__ Z, Vec3d E, int want_f, const double* __restrict__ vel,
           double* __restrict__ fext, double* __restrict__ pdot)
{
    __shared__ double sh[3][8];
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    double pd[3] = {0.0, 0.0, 0.0};
    if (i < N) {
        double z[9];
#pragma unroll
        for (int c = 0; c < 9; ++c) z[c] = Z[(int64_t)c * N + i];
        if (want_f) {
#pragma unroll
            for (int b = 0; b < 3; ++b) fext[(int64_t)b * N + i] = E.v[0] * z[b] + E.v[1] * z[3 + b] + E.v[2] * z[6 + b];   // Eq. 29
        }
        if (vel) {
            const double v0 = vel[i], v1 = vel[N + i], v2 = vel[2 * N + i];
#pragma unroll
            for (int a = 0; a < 3; ++a) pd[a] = z[3 * a] * v0 + z[3 * a + 1] * v1 + z[3 * a + 2] * v2;                      // Eq. 30
        }
    }
    if (vel) {
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            double x = pd[a];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
            if ((threadIdx.x & 31) == 0) sh[a][threadIdx.x >> 5] = x;
        }
        __syncthreads();
        if (threadIdx.x < 3) {
            double r = 0.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) r += sh[threadIdx.x][w];
            atomicAdd(&pdot[threadIdx.x], r);
        }
    }
}

void drop_md_graphs(qnep_handle* h)
{
    for (int k = 0; k < 2; ++k) {
        if (h->md_exec[k]) cudaGraphExecDestroy(h->md_exec[k]);
        h->md_exec[k] = nullptr;
    }
}

int upload_model(qnep_handle* h)
{
    const qnep_model_desc& m = h->model;
    const int T = m.n_types, H = m.n_neurons, D = h->ND;
    const float* p = h->h_params.data();
    const size_t ncoef = (size_t)T * T * QNEP_NRAD * QNEP_NB;
    const float* cR = p;
    const float* cA = cR + ncoef;
    const float* scaler = cA + ncoef;
    const float* nn = scaler + D;
    const int per_type = H * D + 3 * H;
    const float* b1 = nn + (size_t)T * per_type;
    // padded coefficient tables [T*T][5][KPAD]
    std::vector<float> pR((size_t)T * T * QNEP_NRAD * QNEP_KPAD, 0.f), pA(pR.size(), 0.f);
    for (int tt = 0; tt < T * T; ++tt)
        for (int n = 0; n < QNEP_NRAD; ++n)
            for (int k = 0; k < QNEP_NB; ++k) {
                pR[((size_t)tt * QNEP_NRAD + n) * QNEP_KPAD + k] = cR[((size_t)tt * QNEP_NRAD + n) * QNEP_NB + k];
                pA[((size_t)tt * QNEP_NRAD + n) * QNEP_KPAD + k] = cA[((size_t)tt * QNEP_NRAD + n) * QNEP_NB + k];
            }
    // NN per type: w0 * scaler in rows padded to 28, then b0, w1U, w1q
    const int W0P = (D + 3) / 4 * 4;
    h->w0p = W0P;
    h->nn_stride = H * W0P + 3 * H;
    h->nn_stride = (h->nn_stride + 3) / 4 * 4;
    std::vector<float> pn((size_t)T * h->nn_stride, 0.f);
    for (int t = 0; t < T; ++t) {
        const float* src = nn + (size_t)t * per_type;
        float* dst = pn.data() + (size_t)t * h->nn_stride;
        for (int mu = 0; mu < H; ++mu)
            for (int v = 0; v < D; ++v) dst[mu * W0P + v] = src[mu * D + v] * scaler[v];
        for (int i = 0; i < 3 * H; ++i) dst[H * W0P + i] = src[H * D + i];
    }
    h->b1U = b1[0];
    h->b1q = b1[1];
    int rc;
    if ((rc = dev_alloc(h, &h->d_cR, pR.size()))) return rc;
    if ((rc = dev_alloc(h, &h->d_cA, pA.size()))) return rc;
    if ((rc = dev_alloc(h, &h->d_nn, pn.size()))) return rc;
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_cR, pR.data(), sizeof(float) * pR.size(), cudaMemcpyHostToDevice));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_cA, pA.data(), sizeof(float) * pA.size(), cudaMemcpyHostToDevice));
    QNEP_CUDA_OK(h, cudaMemcpy(h->d_nn, pn.data(), sizeof(float) * pn.size(), cudaMemcpyHostToDevice));
    return QNEP_OK;
}

// host-side decision of a pipeline run: does this evaluation rebuild the neighbour list?  (updates the counters)
bool plan_pipeline(qnep_handle* h)
{
    const bool rebuild = h->force_rebuild || h->rebuild_every <= 1 || h->calls_since_build < 0 ||
                         h->calls_since_build >= h->rebuild_every;
    if (rebuild) {
        h->calls_since_build = 0;
        h->force_rebuild = false;
    }
    h->rebuilt_last = rebuild;
    h->calls_since_build += 1;
    return rebuild;
}

// the pipeline proper (enqueue only); `timed` = false leaves out the stage events (stream capture: qnep_md_run's graphs)
int enqueue_pipeline(qnep_handle* h, bool rebuild, bool timed, int64_t N, const double* pos, const int32_t* types, uint32_t want,
                     double* energy, double* forces, double* virial, double* charges, double* bec, cudaStream_t s,
                     double* atom_virial = nullptr)
{
    int rc;
    const bool atomv = (want & QNEP_WANT_ATOM_VIRIAL) && atom_virial;
    if (atomv && !h->d_Wat) QNEP_CUDA_OK(h, cudaMalloc(&h->d_Wat, sizeof(float) * 9 * (size_t)N));
    cudaEvent_t* ev = nullptr;
    if (timed) {
        ev = h->ring.data() + (size_t)(h->prof_count % qnep_handle::RING) * qnep_handle::NEV;
        h->ev = ev;
        h->prof_count += 1;
    }
#define QNEP_STAGE(i) do { if (timed) QNEP_CUDA_OK(h, cudaEventRecord(ev[i], s)); } while (0)
    QNEP_STAGE(0);
    QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_sums, 0, sizeof(double) * QNEP_SUM_ALLOC, s));
    if (rebuild) { if ((rc = qnep_launch_build(h, pos, types, s))) return rc; }
    QNEP_STAGE(1);
    if (!rebuild) { if ((rc = qnep_launch_prep(h, pos, false, s))) return rc; }
    QNEP_STAGE(2);
    if ((rc = qnep_launch_pairs(h, s))) return rc;
    QNEP_STAGE(3);
    if ((rc = qnep_launch_desc_angular(h, s))) return rc;
    QNEP_STAGE(4);
    if ((rc = qnep_launch_nn(h, (want & QNEP_WANT_CHARGES) ? charges : nullptr, s))) return rc;
    if (h->early_q_host && (want & QNEP_WANT_CHARGES)) {
        // qnep_compute_host: the charges are final here (Eq. 33); their device-to-host copy overlaps the rest of the evaluation
        QNEP_CUDA_OK(h, cudaEventRecord(h->ev_q_ready, s));
        QNEP_CUDA_OK(h, cudaStreamWaitEvent(h->copy_stream, h->ev_q_ready, 0));
        QNEP_CUDA_OK(h, cudaMemcpyAsync(h->early_q_host, h->early_q_dev, sizeof(double) * N, cudaMemcpyDeviceToHost, h->copy_stream));
        QNEP_CUDA_OK(h, cudaEventRecord(h->ev_q_copied, h->copy_stream));
    }
    QNEP_STAGE(5);
    if (h->es.method != 0 && h->model.mode == 1) { if ((rc = qnep_launch_realspace(h, atomv, s))) return rc; }
    QNEP_STAGE(6);
    if (h->es.method == 1) { if ((rc = qnep_launch_ewald(h, pos, atomv, s))) return rc; }
    else if (h->es.method == 2) {
        if ((rc = qnep_launch_pppm(h, (want & QNEP_WANT_VIRIAL) != 0, s))) return rc;
        if (atomv) { if ((rc = qnep_launch_pppm_atom_virial(h, s))) return rc; }
    } else {
        QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_Fs, 0, sizeof(float) * 3 * N, s));
        if (atomv) QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_Wat, 0, sizeof(float) * 9 * N, s));
    }
    if ((rc = qnep_launch_phi_finalize(h, s))) return rc;
    const bool need_forces = atomv || (want & (QNEP_WANT_FORCES | QNEP_WANT_VIRIAL)) != 0;
    const bool need_virial = atomv || (want & QNEP_WANT_VIRIAL) != 0;
    QNEP_STAGE(7);
    if (need_forces) {
        if ((rc = qnep_launch_force_angular(h, false, need_virial, atomv, s))) return rc;     // bracketed alone by ev[7], ev[8]
        QNEP_STAGE(8);
        double* fout = ((want & QNEP_WANT_FORCES) && forces) ? forces : h->d_Fmd;
        if ((rc = qnep_launch_force_radial(h, false, need_virial, fout, atomv ? atom_virial : nullptr, s))) return rc;
    } else {
        QNEP_STAGE(8);
    }
    k_finalize<<<1, 32, 0, s>>>(h->d_sums, h->model.mode, (want & QNEP_WANT_ENERGY) ? energy : nullptr,
                                (want & QNEP_WANT_VIRIAL) ? virial : nullptr);
    h->launches += 1;
    QNEP_STAGE(9);
    if ((want & QNEP_WANT_BEC) && bec) {
        if ((rc = qnep_launch_force_angular(h, true, false, false, s))) return rc;
        if ((rc = qnep_launch_force_radial(h, true, false, bec, nullptr, s))) return rc;
    }
    QNEP_STAGE(10);
#undef QNEP_STAGE
    h->ev_valid = timed;
    QNEP_CUDA_OK(h, cudaMemcpyAsync(h->h_flags, h->d_flags, sizeof(int) * FLAG_COUNT, cudaMemcpyDeviceToHost, s));
    if (timed) QNEP_CUDA_OK(h, cudaEventRecord(h->ev_flags, s));
    h->flags_pending = true;
    h->last_stream = s;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int run_pipeline(qnep_handle* h, int64_t N, const double* pos, const int32_t* types, uint32_t want, double* energy,
                 double* forces, double* virial, double* charges, double* bec, cudaStream_t s)
{
    const bool rebuild = plan_pipeline(h);
    return enqueue_pipeline(h, rebuild, true, N, pos, types, want, energy, forces, virial, charges, bec, s);
}

int check_args(qnep_handle* h, int64_t n_atoms, const void* pos, const void* types, const double* box, uint32_t want,
               const void* energy, const void* forces, const void* virial, const void* charges, const void* bec)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (n_atoms <= 0 || n_atoms > QNEP_NL_MASK) { h->err = "n_atoms out of range"; return QNEP_ERR_INVALID_ARG; }
    if (!pos || !types || !box) { h->err = "null input pointer"; return QNEP_ERR_INVALID_ARG; }
    if (((want & QNEP_WANT_ENERGY) && !energy) || ((want & QNEP_WANT_FORCES) && !forces) ||
        ((want & QNEP_WANT_VIRIAL) && !virial) || ((want & QNEP_WANT_CHARGES) && !charges) ||
        ((want & QNEP_WANT_BEC) && !bec)) {
        h->err = "a requested output pointer is null";
        return QNEP_ERR_INVALID_ARG;
    }
    return QNEP_OK;
}

}  // namespace

extern "C" {

int qnep_create(const qnep_model_desc* model, const float* params_host, size_t n_params, const qnep_es_desc* es,
                qnep_handle** out)
{
    if (out) *out = nullptr;
    if (!model || !params_host || !es || !out) { g_create_error = "null argument"; return QNEP_ERR_INVALID_ARG; }
    qnep_handle* h = new (std::nothrow) qnep_handle();
    if (!h) { g_create_error = "out of host memory"; return QNEP_ERR_OOM; }
    auto fail = [&](int code) { g_create_error = h->err; qnep_destroy(h); return code; };
    h->model = *model;
    std::memset(h->box, 0, sizeof(h->box));
    std::memset(&h->geo, 0, sizeof(h->geo));
    const qnep_model_desc& m = h->model;
    if (m.n_types < 1 || m.n_neurons < 1 || m.rc_r <= 0 || m.rc_a <= 0 || m.rc_a > m.rc_r || (m.mode != 1 && m.mode != 2)) {
        h->err = "invalid model description";
        return fail(QNEP_ERR_INVALID_ARG);
    }
    if (m.n_types > QNEP_MAX_TYPES || m.n_max_r != 4 || m.n_max_a != 4 || m.l_max != 4 || m.basis_r != 8 || m.basis_a != 8 ||
        m.n_neurons > 256) {
        h->err = "this version supports n_types <= 4, n_max = 4, l_max = 4, basis = 8, n_neurons <= 256";
        return fail(QNEP_ERR_UNSUPPORTED);
    }
    if (!((m.l_max_4b == 0 && m.l_max_5b == 0) || (m.l_max_4b == 2 && m.l_max_5b == 1))) {
        h->err = "this version takes the 4-/5-body terms both off (0, 0) or both on (l_max_4b = 2, l_max_5b = 1)";
        return fail(QNEP_ERR_UNSUPPORTED);
    }
    h->ND = m.l_max_4b == 2 ? QNEP_NDESC_HB : QNEP_NDESC;
    h->nn_tensor = (h->ND == QNEP_NDESC && m.n_neurons <= 128) ? 2 : 0;      // tcgen05 kernel where it applies (qnep_set_nn_kernel)
    const int T = m.n_types, H = m.n_neurons, D = h->ND;
    const size_t expect = 2 * (size_t)T * T * QNEP_NRAD * QNEP_NB + D + (size_t)T * (H * D + 3 * H) + 2;
    if (n_params != expect) { h->err = "n_params does not match the model description"; return fail(QNEP_ERR_INVALID_ARG); }
    int rc = validate_es(h, es);
    if (rc) return fail(rc);
    h->es = *es;
    h->alpha = es->alpha > 0 ? es->alpha : M_PI / m.rc_r;
    h->h_params.assign(params_host, params_host + n_params);
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) {
        h->err = "no CUDA device: this library has no CPU fallback";
        return fail(QNEP_ERR_CUDA);
    }
    if ((rc = upload_model(h))) return fail(rc);
    if (cudaMalloc(&h->d_sums, sizeof(double) * QNEP_SUM_ALLOC) != cudaSuccess ||
        cudaMalloc(&h->d_flags, sizeof(int) * FLAG_COUNT) != cudaSuccess ||
        cudaMallocHost(&h->h_flags, sizeof(int) * FLAG_COUNT) != cudaSuccess) {
        h->err = "allocation of accumulators failed";
        return fail(QNEP_ERR_OOM);
    }
    cudaMemset(h->d_flags, 0, sizeof(int) * FLAG_COUNT);
    std::memset(h->h_flags, 0, sizeof(int) * FLAG_COUNT);
    cudaEventCreateWithFlags(&h->ev_flags, cudaEventDisableTiming);
    h->ring.resize((size_t)qnep_handle::RING * qnep_handle::NEV);
    for (auto& e : h->ring) cudaEventCreate(&e);
    *out = h;
    return QNEP_OK;
}

int qnep_set_electrostatics(qnep_handle* h, const qnep_es_desc* es)
{
    if (!h || !es) return QNEP_ERR_INVALID_ARG;
    int rc = validate_es(h, es);
    if (rc) return rc;
    h->es = *es;
    h->alpha = es->alpha > 0 ? es->alpha : M_PI / h->model.rc_r;
    std::memset(h->box, 0, sizeof(h->box));   // forces the tables to be rebuilt at the next compute
    h->force_rebuild = true;
    return QNEP_OK;
}

int qnep_set_neighbor_policy(qnep_handle* h, double skin, int32_t rebuild_every)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (skin < 0 || rebuild_every < 0) { h->err = "skin and rebuild_every must be non-negative"; return QNEP_ERR_INVALID_ARG; }
    h->skin = skin;
    h->rebuild_every = rebuild_every;
    h->force_rebuild = true;
    std::memset(h->box, 0, sizeof(h->box));
    return QNEP_OK;
}

int qnep_set_neighbor_capacity(qnep_handle* h, int32_t cap_radial, int32_t cap_angular)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    h->user_capR = cap_radial > 0 ? cap_radial : 0;
    h->user_capLR = h->user_capR;
    h->user_capA = cap_angular > 0 ? cap_angular : 0;
    h->force_rebuild = true;
    return QNEP_OK;
}

int qnep_compute(qnep_handle* h, int64_t n_atoms, const double* pos_dev, const int32_t* types_dev, const double box[9],
                 uint32_t want, double* energy_dev, double* forces_dev, double* virial_dev, double* charges_dev,
                 double* bec_dev, void* cuda_stream)
{
    int rc = check_args(h, n_atoms, pos_dev, types_dev, box, want, energy_dev, forces_dev, virial_dev, charges_dev, bec_dev);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (h->flags_pending && cudaEventQuery(h->ev_flags) == cudaSuccess) {
        if ((rc = consume_flags(h))) return rc;
    }
    if ((rc = ensure_workspace(h, n_atoms, box))) return rc;
    h->md_have_forces = false;
    return run_pipeline(h, n_atoms, pos_dev, types_dev, want, energy_dev, forces_dev, virial_dev, charges_dev, bec_dev, s);
}

int qnep_compute_atom_virial(qnep_handle* h, int64_t n_atoms, const double* pos_dev, const int32_t* types_dev, const double box[9],
                             uint32_t want, double* energy_dev, double* forces_dev, double* virial_dev, double* charges_dev,
                             double* atom_virial_dev, void* cuda_stream)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (!atom_virial_dev) { h->err = "qnep_compute_atom_virial: null output pointer"; return QNEP_ERR_INVALID_ARG; }
    if (want & QNEP_WANT_BEC) { h->err = "qnep_compute_atom_virial: QNEP_WANT_BEC is not available in this call"; return QNEP_ERR_INVALID_ARG; }
    int rc = check_args(h, n_atoms, pos_dev, types_dev, box, want, energy_dev, forces_dev, virial_dev, charges_dev, nullptr);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (h->flags_pending && cudaEventQuery(h->ev_flags) == cudaSuccess) {
        if ((rc = consume_flags(h))) return rc;
    }
    if ((rc = ensure_workspace(h, n_atoms, box))) return rc;
    h->md_have_forces = false;
    const bool rebuild = plan_pipeline(h);
    return enqueue_pipeline(h, rebuild, true, n_atoms, pos_dev, types_dev, want | QNEP_WANT_ATOM_VIRIAL, energy_dev, forces_dev, virial_dev,
                            charges_dev, nullptr, s, atom_virial_dev);
}

int qnep_md_set_outputs(qnep_handle* h, uint32_t want, double* virial_dev, double* charges_dev)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if ((want & ~(uint32_t)(QNEP_WANT_VIRIAL | QNEP_WANT_CHARGES)) || ((want & QNEP_WANT_VIRIAL) && !virial_dev) ||
        ((want & QNEP_WANT_CHARGES) && !charges_dev)) {
        h->err = "qnep_md_set_outputs: only QNEP_WANT_VIRIAL / QNEP_WANT_CHARGES, each with its output pointer";
        return QNEP_ERR_INVALID_ARG;
    }
    h->md_want = want;
    h->md_virial = (want & QNEP_WANT_VIRIAL) ? virial_dev : nullptr;
    h->md_charges = (want & QNEP_WANT_CHARGES) ? charges_dev : nullptr;
    return QNEP_OK;
}

int qnep_md_reset(qnep_handle* h)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    h->md_have_forces = false;
    h->force_rebuild = true;
    return QNEP_OK;
}

int qnep_set_md_graphs(qnep_handle* h, int32_t mode)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (mode < 0 || mode > 2) { h->err = "qnep_set_md_graphs: mode must be 0, 1 or 2"; return QNEP_ERR_INVALID_ARG; }
    h->md_graph_mode = mode;
    return QNEP_OK;
}

int qnep_set_pppm_kernels(qnep_handle* h, int32_t mode)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (mode < 0 || mode > 2) { h->err = "qnep_set_pppm_kernels: mode must be 0, 1 or 2"; return QNEP_ERR_INVALID_ARG; }
    h->pppm_kernels = mode;
    h->ws_generation += 1;      // captured MD graphs hold the old kernels
    return QNEP_OK;
}

int qnep_set_nn_kernel(qnep_handle* h, int32_t mode)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (mode < 0 || mode > 2) { h->err = "qnep_set_nn_kernel: mode must be 0 (FP32 FMA), 1 (mma.sync) or 2 (tcgen05)"; return QNEP_ERR_INVALID_ARG; }
    if (mode == 2 && h->model.n_neurons > 128) { h->err = "qnep_set_nn_kernel: the tcgen05 kernel takes at most 128 hidden neurons"; return QNEP_ERR_UNSUPPORTED; }
    if (mode == 1) {
        // k_nn_mma keeps the split weight tables of all species in shared memory: T (2 HP 36 + 3 HP) floats, opt-in limit 200 KB
        const size_t HP = (size_t)(h->model.n_neurons + 7) / 8 * 8;
        if (sizeof(float) * (size_t)h->model.n_types * (2 * HP * 36 + 3 * HP) > 200 * 1024) {
            h->err = "qnep_set_nn_kernel: the mma.sync kernel's weight tables (n_types x n_neurons) exceed 200 KB of shared memory";
            return QNEP_ERR_UNSUPPORTED;
        }
    }
    if (mode != 0 && h->ND != QNEP_NDESC) { h->err = "qnep_set_nn_kernel: the tensor-core kernel takes the 25-descriptor model only"; return QNEP_ERR_UNSUPPORTED; }
    h->nn_tensor = mode;
    h->ws_generation += 1;      // captured MD graphs hold the old kernel
    h->md_have_forces = false;
    return QNEP_OK;
}

int qnep_set_zbl(qnep_handle* h, int32_t enabled, double r_inner, double r_outer, const double* z_host)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    ZblParams z = {};
    if (enabled) {
        if (!z_host || !(r_inner >= 0.0) || !(r_outer > r_inner)) { h->err = "qnep_set_zbl: need 0 <= r_inner < r_outer and atomic numbers"; return QNEP_ERR_INVALID_ARG; }
        if (r_outer > h->model.rc_a) { h->err = "qnep_set_zbl: r_outer beyond the angular cutoff (the core is evaluated on the angular pair list)"; return QNEP_ERR_UNSUPPORTED; }
        const int T = h->model.n_types;
        for (int t = 0; t < T; ++t)
            if (!(z_host[t] > 0.0)) { h->err = "qnep_set_zbl: atomic numbers must be positive"; return QNEP_ERR_INVALID_ARG; }
        z.on = 1;
        z.r1 = (float)r_inner; z.r2 = (float)r_outer; z.r2sq = (float)(r_outer * r_outer);
        z.sw = (float)(M_PI / (r_outer - r_inner));
        for (int a = 0; a < T; ++a)
            for (int b = 0; b < T; ++b) {
                z.kzz[a][b] = (float)(QNEP_K_COULOMB * z_host[a] * z_host[b]);
                z.ainv[a][b] = (float)((std::pow(z_host[a], 0.23) + std::pow(z_host[b], 0.23)) / 0.46850);
            }
    }
    h->zbl = z;
    h->ws_generation += 1;      // captured MD graphs hold the old kernel arguments
    h->md_have_forces = false;
    return QNEP_OK;
}

int qnep_check(qnep_handle* h)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    QNEP_CUDA_OK(h, cudaStreamSynchronize(h->last_stream));
    QNEP_CUDA_OK(h, cudaGetLastError());
    if (h->flags_pending) return consume_flags(h);
    return QNEP_OK;
}

int qnep_compute_host(qnep_handle* h, int64_t n_atoms, const double* pos_host, const int32_t* types_host,
                      const double box[9], uint32_t want, double* energy_host, double* forces_host, double* virial_host,
                      double* charges_host, double* bec_host, void* cuda_stream)
{
    int rc = check_args(h, n_atoms, pos_host, types_host, box, want, energy_host, forces_host, virial_host, charges_host, bec_host);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)n_atoms;
    const bool fresh = h->hostN != n_atoms;
    if (fresh) {
        if ((rc = dev_alloc(h, &h->d_hpos, 3 * n))) return rc;
        if ((rc = dev_alloc(h, &h->d_htypes, n))) return rc;
        if ((rc = dev_alloc(h, &h->d_hout, 1 + 3 * n + 9 + n + 9 * n))) return rc;
        h->hostN = n_atoms;
    }
    double* d_e = h->d_hout;
    double* d_f = d_e + 1;
    double* d_w = d_f + 3 * n;
    double* d_q = d_w + 9;
    double* d_z = d_q + n;
    QNEP_CUDA_OK(h, cudaMemcpyAsync(h->d_hpos, pos_host, sizeof(double) * 3 * n, cudaMemcpyHostToDevice, s));
    // The species are read by the neighbour build only (between builds they sit in the sorted coordinate array), so they travel
    // only with the calls that can rebuild: same predicate as plan_pipeline / ensure_workspace, erring on the side of copying.
    const bool may_rebuild = fresh || h->force_rebuild || h->rebuild_every <= 1 || h->calls_since_build < 0 ||
                             h->calls_since_build >= h->rebuild_every || h->N != n_atoms || h->flags_pending ||
                             std::memcmp(box, h->box, sizeof(double) * 9) != 0;
    if (may_rebuild) QNEP_CUDA_OK(h, cudaMemcpyAsync(h->d_htypes, types_host, sizeof(int32_t) * n, cudaMemcpyHostToDevice, s));
    const bool early_q = (want & QNEP_WANT_CHARGES) != 0;
    if (early_q) {
        if (!h->copy_stream) {
            QNEP_CUDA_OK(h, cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
            QNEP_CUDA_OK(h, cudaEventCreateWithFlags(&h->ev_q_ready, cudaEventDisableTiming));
            QNEP_CUDA_OK(h, cudaEventCreateWithFlags(&h->ev_q_copied, cudaEventDisableTiming));
        }
        h->early_q_host = charges_host; h->early_q_dev = d_q;
    }
    rc = qnep_compute(h, n_atoms, h->d_hpos, h->d_htypes, box, want, d_e, d_f, d_w, d_q, d_z, s);
    h->early_q_host = nullptr; h->early_q_dev = nullptr;
    if (rc) return rc;
    if (want & QNEP_WANT_ENERGY) QNEP_CUDA_OK(h, cudaMemcpyAsync(energy_host, d_e, sizeof(double), cudaMemcpyDeviceToHost, s));
    if (want & QNEP_WANT_FORCES) QNEP_CUDA_OK(h, cudaMemcpyAsync(forces_host, d_f, sizeof(double) * 3 * n, cudaMemcpyDeviceToHost, s));
    if (want & QNEP_WANT_VIRIAL) QNEP_CUDA_OK(h, cudaMemcpyAsync(virial_host, d_w, sizeof(double) * 9, cudaMemcpyDeviceToHost, s));
    if (early_q) QNEP_CUDA_OK(h, cudaStreamWaitEvent(s, h->ev_q_copied, 0));      // the copy was enqueued inside the pipeline
    if (want & QNEP_WANT_BEC) QNEP_CUDA_OK(h, cudaMemcpyAsync(bec_host, d_z, sizeof(double) * 9 * n, cudaMemcpyDeviceToHost, s));
    return qnep_check(h);
}

int qnep_md_run(qnep_handle* h, int64_t n_atoms, double* pos_dev, double* vel_dev, const int32_t* types_dev,
                const double box[9], const double* mass_host, double dt, int32_t n_steps, double* energy_dev,
                void* cuda_stream)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (n_atoms <= 0 || !pos_dev || !vel_dev || !types_dev || !box || !mass_host || n_steps < 0) {
        h->err = "invalid argument to qnep_md_run";
        return QNEP_ERR_INVALID_ARG;
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int rc;
    if (h->flags_pending) { if ((rc = qnep_check(h))) return rc; }
    if ((rc = ensure_workspace(h, n_atoms, box))) return rc;
    Masses ms;
    for (int t = 0; t < QNEP_MAX_TYPES; ++t) ms.m[t] = t < h->model.n_types ? mass_host[t] : 1.0;
    const int nb = (int)((n_atoms + 255) / 256);
    const uint32_t want = QNEP_WANT_ENERGY | QNEP_WANT_FORCES | h->md_want;
    double* const mdW = h->md_virial;
    double* const mdQ = h->md_charges;
    if (!h->md_have_forces) {
        if ((rc = run_pipeline(h, n_atoms, pos_dev, types_dev, want, nullptr, h->d_Fmd, mdW, mdQ, nullptr, s))) return rc;
        h->md_have_forces = true;
    }
    const bool graphs = h->md_graph_mode == 2 || (h->md_graph_mode == 1 && n_atoms <= QNEP_GRAPH_MAX_ATOMS);
    cudaStream_t caller = s;
    if (graphs && n_steps > 0) {
        // the steps run on the handle's own stream, after everything the caller has enqueued so far
        if (!h->md_stream) {
            QNEP_CUDA_OK(h, cudaStreamCreateWithFlags(&h->md_stream, cudaStreamNonBlocking));
            QNEP_CUDA_OK(h, cudaEventCreateWithFlags(&h->md_fence, cudaEventDisableTiming));
        }
        QNEP_CUDA_OK(h, cudaEventRecord(h->md_fence, caller));
        QNEP_CUDA_OK(h, cudaStreamWaitEvent(h->md_stream, h->md_fence, 0));
        s = h->md_stream;
    }
    if (graphs && n_steps > 0) {
        qnep_handle::MdKey key = {};
        key.pos = pos_dev; key.vel = vel_dev; key.types = types_dev; key.N = n_atoms; key.dt = dt; key.s = nullptr;     // replay always happens on md_stream
        key.virial = mdW; key.charges = mdQ; key.want = want;
        key.gen = h->ws_generation;
        for (int t = 0; t < QNEP_MAX_TYPES; ++t) key.m[t] = ms.m[t];
        if (std::memcmp(&key, &h->md_key, sizeof(key)) != 0) {
            drop_md_graphs(h);
            h->md_key = key;
        }
    }
    for (int step = 0; step < n_steps; ++step) {
        if (!graphs) {
            k_vv_kick_drift<<<nb, 256, 0, s>>>(n_atoms, pos_dev, vel_dev, h->d_Fmd, types_dev, ms, dt);
            if ((rc = run_pipeline(h, n_atoms, pos_dev, types_dev, want, nullptr, h->d_Fmd, mdW, mdQ, nullptr, s))) return rc;
            k_vv_kick<<<nb, 256, 0, s>>>(n_atoms, vel_dev, h->d_Fmd, types_dev, ms, dt, h->d_sums);
            h->launches += 2;
            continue;
        }
        const int kind = plan_pipeline(h) ? 1 : 0;
        if (!h->md_exec[kind]) {
            // capture one step of this kind; nothing runs until the graph is launched below
            const int64_t l0 = h->launches;
            cudaGraph_t graph = nullptr;
            QNEP_CUDA_OK(h, cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal));
            k_vv_kick_drift<<<nb, 256, 0, s>>>(n_atoms, pos_dev, vel_dev, h->d_Fmd, types_dev, ms, dt);
            rc = enqueue_pipeline(h, kind == 1, false, n_atoms, pos_dev, types_dev, want, nullptr, h->d_Fmd, mdW, mdQ, nullptr, s);
            k_vv_kick<<<nb, 256, 0, s>>>(n_atoms, vel_dev, h->d_Fmd, types_dev, ms, dt, h->d_sums);
            const cudaError_t ce = cudaStreamEndCapture(s, &graph);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            QNEP_CUDA_OK(h, ce);
            const cudaError_t ci = cudaGraphInstantiate(&h->md_exec[kind], graph, 0);
            cudaGraphDestroy(graph);
            QNEP_CUDA_OK(h, ci);
            h->md_exec_launches[kind] = h->launches - l0 + 2;
            h->launches = l0;
        }
        QNEP_CUDA_OK(h, cudaGraphLaunch(h->md_exec[kind], s));
        h->launches += h->md_exec_launches[kind];
        h->ev_valid = false;
        h->flags_pending = true;
        h->last_stream = s;
    }
    if (s != caller) {
        // hand back to the caller's stream
        QNEP_CUDA_OK(h, cudaEventRecord(h->md_fence, s));
        QNEP_CUDA_OK(h, cudaStreamWaitEvent(caller, h->md_fence, 0));
        s = caller;
        h->last_stream = caller;
    }
    if (energy_dev) { k_md_energy<<<1, 1, 0, s>>>(h->d_sums, h->model.mode, energy_dev); h->launches += 1; }
    return qnep_check(h);
}

int qnep_get_timings(qnep_handle* h, float* ms, int32_t n)
{
    if (!h || !ms) return QNEP_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) ms[i] = 0.f;
    if (!h->ev_valid) return QNEP_OK;
    QNEP_CUDA_OK(h, cudaEventSynchronize(h->ev[10]));
    // ev[i] .. ev[i+1] -> stage i
    for (int i = 0; i < QNEP_T_TOTAL && i < n; ++i) {
        float t = 0.f;
        QNEP_CUDA_OK(h, cudaEventElapsedTime(&t, h->ev[i], h->ev[i + 1]));
        ms[i] = t;
    }
    if (n > QNEP_T_TOTAL) {
        float t = 0.f;
        QNEP_CUDA_OK(h, cudaEventElapsedTime(&t, h->ev[0], h->ev[10]));
        ms[QNEP_T_TOTAL] = t;
    }
    return QNEP_OK;
}

int qnep_profile_reset(qnep_handle* h)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    h->prof_count = 0;
    return QNEP_OK;
}

int qnep_profile_sum(qnep_handle* h, float* ms, int32_t n, int64_t* n_evals)
{
    if (!h || !ms || !n_evals) return QNEP_ERR_INVALID_ARG;
    for (int i = 0; i < n; ++i) ms[i] = 0.f;
    const int64_t cnt = std::min<int64_t>(h->prof_count, qnep_handle::RING);
    *n_evals = cnt;
    if (cnt == 0) return QNEP_OK;
    QNEP_CUDA_OK(h, cudaStreamSynchronize(h->last_stream));
    for (int64_t c = 0; c < cnt; ++c) {
        const int64_t slot = (h->prof_count - 1 - c) % qnep_handle::RING;
        cudaEvent_t* ev = h->ring.data() + (size_t)slot * qnep_handle::NEV;
        for (int i = 0; i < QNEP_T_TOTAL && i < n; ++i) {
            float t = 0.f;
            QNEP_CUDA_OK(h, cudaEventElapsedTime(&t, ev[i], ev[i + 1]));
            ms[i] += t;
        }
        if (n > QNEP_T_TOTAL) {
            float t = 0.f;
            QNEP_CUDA_OK(h, cudaEventElapsedTime(&t, ev[0], ev[QNEP_T_TOTAL]));
            ms[QNEP_T_TOTAL] += t;
        }
    }
    return QNEP_OK;
}

int qnep_response(qnep_handle* h, int64_t n_atoms, const double* bec_dev, const double* efield_host, const double* vel_dev,
                  double* fext_dev, double* pdot_dev, void* cuda_stream)
{
    if (!h) return QNEP_ERR_INVALID_ARG;
    if (n_atoms <= 0 || !bec_dev) { h->err = "qnep_response: n_atoms <= 0 or null BEC pointer"; return QNEP_ERR_INVALID_ARG; }
    if ((efield_host && !fext_dev) || (vel_dev && !pdot_dev)) { h->err = "qnep_response: a requested output pointer is null"; return QNEP_ERR_INVALID_ARG; }
    if (!efield_host && !vel_dev) return QNEP_OK;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    Vec3d E = {{0.0, 0.0, 0.0}};
    if (efield_host) for (int a = 0; a < 3; ++a) E.v[a] = efield_host[a];
    if (vel_dev) QNEP_CUDA_OK(h, cudaMemsetAsync(pdot_dev, 0, sizeof(double) * 3, s));
    const int nb = (int)((n_atoms + 255) / 256);
    k_response<<<nb, 256, 0, s>>>(n_atoms, bec_dev, E, efield_host ? 1 : 0, vel_dev, fext_dev, pdot_dev);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int64_t qnep_kernel_launches(const qnep_handle* h) { return h ? h->launches : 0; }

int qnep_abi_version(void) { return QNEP_ABI_VERSION; }

int qnep_neighbor_stats(qnep_handle* h, double out[6])
{
    if (!h || !out) return QNEP_ERR_INVALID_ARG;
    for (int i = 0; i < 6; ++i) out[i] = 0;
    if (!h->d_flags || h->N == 0) return QNEP_OK;
    return qnep_launch_list_stats(h, out, h->last_stream);
}

int qnep_fma_peak(double* tflops_host, void* cuda_stream)
{
    if (!tflops_host) return QNEP_ERR_INVALID_ARG;
    return qnep_launch_fma_peak(tflops_host, (cudaStream_t)cuda_stream);
}

int qnep_debug_copy(qnep_handle* h, int32_t which, double* dst, int64_t n)
{
    if (!h || !dst || h->N == 0) return QNEP_ERR_INVALID_ARG;
    const int64_t N = h->N;
    cudaStream_t s = h->last_stream;
    const int nb = (int)((N + 255) / 256);
    auto need = [&](int64_t cnt) { if (n < cnt) { h->err = "debug buffer too small"; return false; } return true; };
    switch (which) {
        case QNEP_DBG_DESCRIPTORS: if (!need(N * h->ND)) return QNEP_ERR_INVALID_ARG;
            k_dbg_rows<<<nb, 256, 0, s>>>(N, h->ND, h->d_D, h->d_sidx, 1, dst); break;
        case QNEP_DBG_SITE_ENERGY: if (!need(N)) return QNEP_ERR_INVALID_ARG;
            k_dbg_rows<<<nb, 256, 0, s>>>(N, 1, h->d_Ui, h->d_sidx, 1, dst); break;
        case QNEP_DBG_Q_RAW: if (!need(N)) return QNEP_ERR_INVALID_ARG;
            k_dbg_rows<<<nb, 256, 0, s>>>(N, 1, h->d_qraw, h->d_sidx, 1, dst); break;
        case QNEP_DBG_PHI: if (!need(N)) return QNEP_ERR_INVALID_ARG;
            k_dbg_rows<<<nb, 256, 0, s>>>(N, 1, h->d_phi, h->d_sidx, 1, dst); break;
        case QNEP_DBG_FP: if (!need(N * h->ND)) return QNEP_ERR_INVALID_ARG;
            k_dbg_rows<<<nb, 256, 0, s>>>(N, h->ND, h->d_Fp, h->d_sidx, 1, dst); break;
        case QNEP_DBG_F_STATIC: if (!need(3 * N)) return QNEP_ERR_INVALID_ARG;
            k_dbg_rows<<<nb, 256, 0, s>>>(N, 3, h->d_Fs, h->d_sidx, 0, dst); break;
        case QNEP_DBG_MESH_RHO:
            if (h->es.method != 2 || !h->d_mesh || !need(h->ngrid)) { h->err = "no PPPM mesh"; return QNEP_ERR_INVALID_ARG; }
            k_dbg_copy<<<(int)((h->ngrid + 255) / 256), 256, 0, s>>>(h->ngrid, h->d_mesh, dst); break;
        case QNEP_DBG_ENERGY_PARTS: if (!need(4)) return QNEP_ERR_INVALID_ARG;
            k_dbg_energy<<<1, 1, 0, s>>>(h->d_sums, dst); break;
        default: h->err = "unknown debug selector"; return QNEP_ERR_INVALID_ARG;
    }
    QNEP_CUDA_OK(h, cudaGetLastError());
    QNEP_CUDA_OK(h, cudaStreamSynchronize(s));
    return QNEP_OK;
}

void qnep_destroy(qnep_handle* h)
{
    if (!h) return;
    drop_md_graphs(h);
    if (h->md_stream) cudaStreamDestroy(h->md_stream);
    if (h->copy_stream) { cudaStreamDestroy(h->copy_stream); cudaEventDestroy(h->ev_q_ready); cudaEventDestroy(h->ev_q_copied); }
    if (h->md_fence) cudaEventDestroy(h->md_fence);
    free_workspace(h);
    void* ptrs[] = {h->d_params, h->d_cR, h->d_cA, h->d_nn, h->d_cnt, h->d_start, h->d_fill, h->d_scantmp, h->d_ctot, h->d_cstart, h->d_mbcnt, h->d_mbstart, h->d_mbfill, h->d_sums, h->d_flags, h->d_kvec,
                    h->d_kint, h->d_ephase, h->d_S, h->d_mesh, h->d_half, h->d_cm1, h->d_cm2, h->d_cm3, h->d_Wat, h->d_field, h->d_gtab, h->d_twiddle, h->d_hpos,
                    h->d_htypes, h->d_hout};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (h->h_flags) cudaFreeHost(h->h_flags);
    if (h->ev_flags) cudaEventDestroy(h->ev_flags);
    for (auto& e : h->ring) if (e) cudaEventDestroy(e);
    delete h;
}

const char* qnep_last_error(const qnep_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
