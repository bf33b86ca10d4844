// neighbor.cu -- step a1 of SURVEY.md 8(a): cell list, (type, cell)-sorted atom order and the
// skin neighbour list with image codes (PAPER.md :91, Eq. 13), plus the per-step
// "prep" pass that turns fp64 positions into cell-relative fp32 coordinates.
//
// Layout decisions:
//  * atoms are reordered by key = type * ncells + cell, so a warp holds atoms of ONE species
//    (weights / coefficients become warp-uniform) that are close in space (gathers hit L1/L2);
//  * positions are stored as float4 (x, y, z relative to the atom's own cell origin, type bits):
//    r_ij = off_j - off_i + delta_cell * hcell is formed from small numbers, so fp32 keeps
//    ~1e-7 A resolution in a 217 A box;
//  * a neighbour entry packs the sorted index of j (26 bits) and the cell offset of the image (three signed
//    2-bit fields): the same atom may appear more than once through different images when the box is smaller
//    than 2 (r_c + skin);
//  * lists are column-major [slot][atom] so that a warp reads consecutive words.
#include "qnep_internal.cuh"

namespace {

__device__ __forceinline__ int pack3(int a, int b, int c) { return a | (b << 10) | (c << 20); }

// Position of an atom relative to the origin of search cell c, for any cell (rows of g.h): with the fractional
// coordinate f = r h^-1 and the cell origin c_a / ncell_a,  s_a = f_a - c_a / ncell_a  is wrapped to the periodic image
// nearest to ref_a (0 at build time: nearest to the cell origin; the build-time value on list-reuse steps), and the
// Cartesian offset is d = s h.  fr[a] = c_a / ncell_a + s_a is the (unwrapped) fractional coordinate the PPPM mesh uses.
__device__ __forceinline__ void cell_relative(const Geometry& g, const double r[3], const int c[3], const double ref[3],
                                              double d[3], double fr[3])
{
    double sfr[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double f = r[0] * g.hinv[a] + r[1] * g.hinv[3 + a] + r[2] * g.hinv[6 + a];
        const double org = (double)c[a] / (double)g.ncell[a];
        double sa = f - org;
        sa -= rint(sa - ref[a]);
        sfr[a] = sa;
        fr[a] = org + sa;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) d[k] = sfr[0] * g.h[k] + sfr[1] * g.h[3 + k] + sfr[2] * g.h[6 + k];
}

// PPPM mesh coordinate (reading S10) of fractional coordinate f on an axis of n points: nearest mesh point i0 (wrapped
// into 0..n-1) and the offset from it in mesh units
__device__ __forceinline__ void mesh_coord(double f, int n, float* frac, int* i0)
{
    const double u = f * n;
    const double r = floor(u + 0.5);
    *frac = (float)(u - r);
    const int ir = (int)r % n;
    *i0 = ir < 0 ? ir + n : ir;
}

// ---- binning -------------------------------------------------------------------------------
__global__ void k_bin_count(int64_t N, int T, const double* __restrict__ pos, const int32_t* __restrict__ types,
                            Geometry g, int* __restrict__ key, int* __restrict__ cnt, int* __restrict__ flags)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int c[3];
    const double r[3] = {pos[i], pos[N + i], pos[2 * N + i]};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        double f = r[0] * g.hinv[a] + r[1] * g.hinv[3 + a] + r[2] * g.hinv[6 + a];
        f -= floor(f);
        int ci = (int)(f * g.ncell[a]);
        c[a] = min(max(ci, 0), g.ncell[a] - 1);
    }
    int cell = (c[0] * g.ncell[1] + c[1]) * g.ncell[2] + c[2];
    int t = types[i];
    if (t < 0 || t >= T) { atomicOr(&flags[FLAG_BAD_TYPE], 1); t = 0; }      // reported as INVALID_ARG; nothing is written out of bounds
    int k = t * g.ncells + cell;
    key[i] = k;
    atomicAdd(&cnt[k], 1);
}

// single-block exclusive scan over n ints (n up to a few million; runs once per rebuild)
__global__ void k_exclusive_scan(int n, const int* __restrict__ in, int* __restrict__ out)
{
    __shared__ int warp_sums[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int base = 0; base < n; base += blockDim.x) {
        int idx = base + threadIdx.x;
        int v = idx < n ? in[idx] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) warp_sums[wid] = x;
        __syncthreads();
        if (wid == 0) {
            int w = lane < (blockDim.x >> 5) ? warp_sums[lane] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += y;
            }
            warp_sums[lane] = w;
        }
        __syncthreads();
        int prefix = carry + (wid > 0 ? warp_sums[wid - 1] : 0) + x - v;
        if (idx < n) out[idx] = prefix;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry = prefix + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) out[n] = carry;
}

// Exclusive scan over many blocks (key counts grow with the volume: T x ncells): every block scans SCAN_CHUNK elements in
// place and reports its total, the totals are scanned by the single-block kernel above, a third pass adds the offsets.
constexpr int SCAN_CHUNK = 2048;      // two elements per thread of a 1024-thread block

__global__ void __launch_bounds__(1024)
k_scan_chunks(int n, const int* __restrict__ in, int* __restrict__ out, int* __restrict__ totals)
{
    __shared__ int warp_sums[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int i0 = blockIdx.x * SCAN_CHUNK + 2 * threadIdx.x;
    const int a = i0 < n ? in[i0] : 0, b = i0 + 1 < n ? in[i0 + 1] : 0;
    int x = a + b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
        int w = warp_sums[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += y;
        }
        warp_sums[lane] = w;
    }
    __syncthreads();
    const int excl = (wid > 0 ? warp_sums[wid - 1] : 0) + x - (a + b);
    if (i0 < n) out[i0] = excl;
    if (i0 + 1 < n) out[i0 + 1] = excl + a;
    if (threadIdx.x == 1023) totals[blockIdx.x] = excl + a + b;
}

__global__ void k_scan_add(int n, int* __restrict__ out, const int* __restrict__ offsets, int nchunks)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] += offsets[i / SCAN_CHUNK];
    if (i == n) out[n] = offsets[nchunks];        // grand total behind the last element
}

// out[0 .. n] = exclusive scan of in[0 .. n-1] (out[n] = total); tmp holds 2 (nchunks + 1) ints
static void exclusive_scan(int n, const int* in, int* out, int* tmp, cudaStream_t s)
{
    if (n <= 4 * SCAN_CHUNK) { k_exclusive_scan<<<1, 1024, 0, s>>>(n, in, out); return; }
    const int nchunks = (n + SCAN_CHUNK - 1) / SCAN_CHUNK;
    k_scan_chunks<<<nchunks, 1024, 0, s>>>(n, in, out, tmp);
    k_exclusive_scan<<<1, 1024, 0, s>>>(nchunks, tmp, tmp + nchunks + 1);
    k_scan_add<<<(n + 1 + 255) / 256, 256, 0, s>>>(n, out, tmp + nchunks + 1, nchunks);
}

__global__ void k_scatter(int64_t N, const int* __restrict__ key, const int* __restrict__ start,
                          int* __restrict__ fill, int* __restrict__ tmpidx)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int k = key[i];
    int slot = start[k] + atomicAdd(&fill[k], 1);
    tmpidx[slot] = (int)i;
}

// deterministic order inside a bucket: rank by original index
__global__ void k_rank(int64_t N, const int* __restrict__ key, const int* __restrict__ start,
                       const int* __restrict__ tmpidx, int* __restrict__ sidx)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    int me = tmpidx[p];
    int k = key[me];
    int b = start[k], e = start[k + 1];
    int rank = 0;
    for (int q = b; q < e; ++q) rank += (tmpidx[q] < me);
    sidx[b + rank] = me;
}

// ---- cell-major order for the PPPM kernels ---------------------------------------------------------
// The neighbour kernels want a warp to hold ONE species, hence the (type, cell) order.  Spreading and back-
// interpolation want atoms that are close in space to be close in the launch order whatever their species, so that
// the mesh is swept once: rank q = cstart[cell] + (atoms of lower species in the cell) + (rank inside the bucket).
__global__ void k_cell_totals(int ncells, int T, const int* __restrict__ cnt, int* __restrict__ ctot)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncells) return;
    int v = 0;
    for (int t = 0; t < T; ++t) v += cnt[t * ncells + c];
    ctot[c] = v;
}

__global__ void k_cm_rank(int64_t N, int ncells, const int* __restrict__ key, const int* __restrict__ sidx,
                          const int* __restrict__ start, const int* __restrict__ cnt, const int* __restrict__ cstart,
                          int* __restrict__ cm, int* __restrict__ cmi)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int k = key[sidx[p]];
    const int t = k / ncells, c = k - t * ncells;
    int q = cstart[c] + ((int)p - start[k]);
    for (int u = 0; u < t; ++u) q += cnt[u * ncells + c];
    cm[p] = q;
    cmi[q] = (int)p;
}

// ---- mesh-bin order for the PPPM kernels (PPPM runs) -------------------------------------------------
// The spreading and back-interpolation kernels (pppm_sweep.cu) work on bins of QNEP_MB_X x QNEP_MB_Y x QNEP_MB_Z mesh
// points: an atom belongs to the bin of its nearest mesh point at BUILD time.  Bins are numbered column by column,
// key = (by * nbz + bz) * nbx + bx, so the atoms a block meets while it sweeps a (y, z) column along x are contiguous.
// q = mbstart[key] + (rank of the sorted index inside the bin) replaces the cell-major rank: cm[p] = q, cmi[q] = p.
__global__ void k_mbin_key(int64_t N, const double* __restrict__ pos, const int* __restrict__ sidx, const int* __restrict__ key,
                           Geometry g, int nbx, int nbz, int* __restrict__ mbkey, int* __restrict__ mbcnt)
{
    const int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const int i = sidx[p];
    const int k = key[i];
    const int cell = k % g.ncells;
    const int c[3] = {cell / (g.ncell[2] * g.ncell[1]), (cell / g.ncell[2]) % g.ncell[1], cell % g.ncell[2]};
    int m0[3];
    {
        const double r[3] = {pos[i], pos[N + i], pos[2 * N + i]}, ref[3] = {0.0, 0.0, 0.0};
        double d[3], ff[3];
        cell_relative(g, r, c, ref, d, ff);                                      // exactly what k_prep does at build time
#pragma unroll
        for (int a = 0; a < 3; ++a) { float fr; mesh_coord(ff[a], g.grid[a], &fr, &m0[a]); }
    }
    const int kb = ((m0[1] / QNEP_MB_Y) * nbz + m0[2] / QNEP_MB_Z) * nbx + m0[0] / QNEP_MB_X;
    mbkey[p] = kb;
    atomicAdd(&mbcnt[kb], 1);
}

__global__ void k_invert_perm(int64_t N, const int* __restrict__ cmi, int* __restrict__ cm)
{
    const int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (q < N) cm[cmi[q]] = (int)q;
}

// ---- per-step prep: cell-relative fp32 coordinates, PPPM mesh coordinates, skin check --------
__global__ void k_prep(int64_t N, const double* __restrict__ pos, const int32_t* __restrict__ types_or_null,
                       const int* __restrict__ sidx, const int* __restrict__ key, const int* __restrict__ cm, Geometry g, int at_build,
                       int* __restrict__ cellc, float4* __restrict__ xyzt, float4* __restrict__ off0,
                       float4* __restrict__ mfrac, int* __restrict__ mi0, int* __restrict__ flags)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    int i = sidx[p];
    int c[3];
    int type;
    if (at_build) {
        int k = key[i];
        type = k / g.ncells;
        int cell = k - type * g.ncells;
        c[2] = cell % g.ncell[2];
        c[1] = (cell / g.ncell[2]) % g.ncell[1];
        c[0] = cell / (g.ncell[2] * g.ncell[1]);
        cellc[p] = pack3(c[0], c[1], c[2]);
    } else {
        int pc = cellc[p];
        c[0] = pc & 1023; c[1] = (pc >> 10) & 1023; c[2] = (pc >> 20) & 1023;
        type = __float_as_int(xyzt[p].w);
    }
    float off[3], dx[3];
    int m0[3];
    // On list-reuse steps the image is the one nearest to the build-time offset, not to the cell origin: with fewer
    // than three cells along an axis an atom near the +-L/2 plane would otherwise flip by a whole L between two steps
    // (a spurious skin violation, and a wrong r_ij for the list built from the other image).
    float o0[3] = {0.f, 0.f, 0.f};
    double ref[3] = {0.0, 0.0, 0.0};
    if (!at_build) {
        const float4 o = off0[p];
        o0[0] = o.x; o0[1] = o.y; o0[2] = o.z;
#pragma unroll
        for (int a = 0; a < 3; ++a) ref[a] = (double)o.x * g.hinv[a] + (double)o.y * g.hinv[3 + a] + (double)o.z * g.hinv[6 + a];
    }
    {
        const double r[3] = {pos[i], pos[N + i], pos[2 * N + i]};
        double d[3], ff[3];
        cell_relative(g, r, c, ref, d, ff);
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            off[a] = (float)d[a];
            if (g.grid[a] > 0) mesh_coord(ff[a], g.grid[a], &dx[a], &m0[a]);
            else { dx[a] = 0.f; m0[a] = 0; }
        }
    }
    float4 v = make_float4(off[0], off[1], off[2], __int_as_float(type));
    xyzt[p] = v;
    {
        const int q = cm[p];                       // PPPM arrays are kept in cell-major order
        mfrac[q] = make_float4(dx[0], dx[1], dx[2], __int_as_float(pack3(m0[0], m0[1], m0[2])));    // w: the packed nearest mesh point (= mi0[q])
        mi0[q] = pack3(m0[0], m0[1], m0[2]);
    }
    if (at_build) {
        off0[p] = v;
    } else {
        float ddx = off[0] - o0[0], ddy = off[1] - o0[1], ddz = off[2] - o0[2];
        if (ddx * ddx + ddy * ddy + ddz * ddz > g.skin_half2) atomicOr(&flags[FLAG_SKIN], 1);
    }
}

// ---- skin neighbour list -----------------------------------------------------------------------
// every (j, image) with r < rc_r + skin; the exact per-step lists are derived from it by k_pairs.
// Warp-tiled int4 layout (qnep_internal.cuh); entries are appended one 4-byte word at a time (the partial vectors
// merge in L2), readers never look beyond the count.  The candidate loop is the whole cost of a rebuild
// (~920 candidates per atom), so it is kept to a dozen instructions per candidate.
__global__ void __launch_bounds__(128)
k_build_lists(int64_t N, int T, Geometry g, const float4* __restrict__ xyzt, const int* __restrict__ cellc,
              const int* __restrict__ start, int capR, int4* __restrict__ nlR, int* __restrict__ nnR,
              int* __restrict__ nnR0, int* __restrict__ nlRend, int* __restrict__ flags)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (p >= N) return;
    const float4 xi = xyzt[p];
    const int ti = __float_as_int(xi.w);
    const int pc = cellc[p];
    const int c0 = pc & 1023, c1 = (pc >> 10) & 1023, c2 = (pc >> 20) & 1023;
    int* out = reinterpret_cast<int*>(nlR + qnep_tiled_base(p, capR / 4));    // slot s at out[(s >> 2) * 128 + (s & 3)]
    int nR = 0, nPad = 0;                // slots written, filler slots among them
    const float rcs2 = g.rcs_r2;
    const float h0 = (float)g.hcell[0], h1 = (float)g.hcell[1], h2 = (float)g.hcell[2];
    const CellVecs cv = qnep_cell_vecs(g.cellv, g.triclinic);
    // type-major order: all neighbours of species 0 first, then species 1, ...  The per-step lists derived from
    // this one inherit the order, so the radial force kernel switches its own coefficient vector T - 1 times per atom.
    for (int t = 0; t < T; ++t) {
        for (int code = 0; code < 27; ++code) {
            const int d0 = code / 9 - 1, d1 = (code / 3) % 3 - 1, d2 = code % 3 - 1;
            // the whole cell is out of reach of this atom?  (positions are relative to the atom's own cell, in [0, hcell);
            // with a single cell along an axis the coordinate is the nearest image to the origin instead: no pruning there)
            if (!g.triclinic) {     // (the gaps along non-orthogonal axes do not add in quadrature: no pruning there)
                const float ex = g.ncell[0] < 2 ? 0.f : (d0 < 0 ? xi.x : (d0 > 0 ? h0 - xi.x : 0.f));
                const float ey = g.ncell[1] < 2 ? 0.f : (d1 < 0 ? xi.y : (d1 > 0 ? h1 - xi.y : 0.f));
                const float ez = g.ncell[2] < 2 ? 0.f : (d2 < 0 ? xi.z : (d2 > 0 ? h2 - xi.z : 0.f));
                const float em = fmaxf(ex, 0.f) * fmaxf(ex, 0.f) + fmaxf(ey, 0.f) * fmaxf(ey, 0.f) + fmaxf(ez, 0.f) * fmaxf(ez, 0.f);
                if (em > rcs2 * 1.0001f) continue;
            }
            int n0 = c0 + d0, n1 = c1 + d1, n2 = c2 + d2;
            n0 = n0 < 0 ? n0 + g.ncell[0] : (n0 >= g.ncell[0] ? n0 - g.ncell[0] : n0);
            n1 = n1 < 0 ? n1 + g.ncell[1] : (n1 >= g.ncell[1] ? n1 - g.ncell[1] : n1);
            n2 = n2 < 0 ? n2 + g.ncell[2] : (n2 >= g.ncell[2] ? n2 - g.ncell[2] : n2);
            const int cell = (n0 * g.ncell[1] + n1) * g.ncell[2] + n2;
            // r_ij = x_j - (x_i - shift)
            float ox = xi.x, oy = xi.y, oz = xi.z;
            {
                float sx = 0.f, sy = 0.f, sz = 0.f;
                qnep_add_image_shift(qnep_image_bits(d0, d1, d2), cv, sx, sy, sz);
                ox -= sx; oy -= sy; oz -= sz;
            }
            const int k = t * g.ncells + cell;
            const int b = start[k], e = start[k + 1];
            const int self = (code == 13 && t == ti) ? (int)p : -1;
            const int cbits = qnep_image_bits(d0, d1, d2);
            auto test = [&](int q, const float4& xj) {
                const float dx = xj.x - ox, dy = xj.y - oy, dz = xj.z - oz;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                if (r2 < rcs2 && q != self) {
                    if (nR < capR) out[((nR >> 2) << 7) | (nR & 3)] = q | cbits;
                    ++nR;
                }
            };
            int q = b;
            for (; q + 4 <= e; q += 4) {
                const float4 x0 = xyzt[q], x1 = xyzt[q + 1], x2 = xyzt[q + 2], x3 = xyzt[q + 3];
                test(q, x0); test(q + 1, x1); test(q + 2, x2); test(q + 3, x3);
            }
            for (; q < e; ++q) test(q, xyzt[q]);
        }
        // Every species segment is padded to a multiple of four slots (one int4) with the atom itself in its own cell
        // (r = 0: the per-step filter drops it), so that the four slots of a list vector belong to ONE species and
        // the walkers decide species, bounds and prefetch once per vector.
        while (nR & 3) {
            if (nR < capR) out[((nR >> 2) << 7) | (nR & 3)] = (int)p;      // zero cell offset
            ++nR; ++nPad;
        }
        nlRend[(int64_t)t * N + p] = min(nR, capR);
    }
    nnR[p] = min(nR, capR);
    nnR0[p] = min(nR, capR) - nPad;
    if (nR > capR) atomicMax(&flags[FLAG_MAX_NR], nR);
}

// max and sum of a per-atom count array (statistics on request only)
__global__ void k_count_stats(int64_t N, const int* __restrict__ cnt, int* __restrict__ out_max,
                              unsigned long long* __restrict__ out_sum)
{
    int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    int v = p < N ? cnt[p] : 0, m = v;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v += __shfl_xor_sync(0xffffffffu, v, o);
        m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    }
    if ((threadIdx.x & 31) == 0) { atomicAdd(out_sum, (unsigned long long)v); atomicMax(out_max, m); }
}

}  // namespace

int qnep_launch_prep(qnep_handle* h, const double* pos, bool at_build, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 255) / 256);
    k_prep<<<nb, 256, 0, s>>>(N, pos, nullptr, h->d_sidx, h->d_key, h->d_cm, h->geo, at_build ? 1 : 0, h->d_cellc, h->d_xyzt,
                              h->d_off0, h->d_mfrac, h->d_mi0, h->d_flags);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

int qnep_launch_build(qnep_handle* h, const double* pos, const int32_t* types, cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 255) / 256);
    QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_cnt, 0, sizeof(int) * (h->nkeys + 1), s));
    QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_fill, 0, sizeof(int) * h->nkeys, s));
    k_bin_count<<<nb, 256, 0, s>>>(N, h->model.n_types, pos, types, h->geo, h->d_key, h->d_cnt, h->d_flags);
    exclusive_scan(h->nkeys, h->d_cnt, h->d_start, h->d_scantmp, s);
    k_scatter<<<nb, 256, 0, s>>>(N, h->d_key, h->d_start, h->d_fill, h->d_tmpidx);
    k_rank<<<nb, 256, 0, s>>>(N, h->d_key, h->d_start, h->d_tmpidx, h->d_sidx);
    if (h->nmbins > 0) {
        // PPPM: mesh-bin order (the sorted index p plays the role of the atom index in k_scatter / k_rank)
        QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_mbcnt, 0, sizeof(int) * (h->nmbins + 1), s));
        QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_mbfill, 0, sizeof(int) * h->nmbins, s));
        k_mbin_key<<<nb, 256, 0, s>>>(N, pos, h->d_sidx, h->d_key, h->geo, h->nmb[0], h->nmb[2], h->d_mbkey, h->d_mbcnt);
        exclusive_scan(h->nmbins, h->d_mbcnt, h->d_mbstart, h->d_scantmp, s);
        k_scatter<<<nb, 256, 0, s>>>(N, h->d_mbkey, h->d_mbstart, h->d_mbfill, h->d_tmpidx);
        k_rank<<<nb, 256, 0, s>>>(N, h->d_mbkey, h->d_mbstart, h->d_tmpidx, h->d_cmi);
        k_invert_perm<<<nb, 256, 0, s>>>(N, h->d_cmi, h->d_cm);
        h->launches += 5;
    } else {
        const int nc = h->geo.ncells;
        k_cell_totals<<<(nc + 255) / 256, 256, 0, s>>>(nc, h->model.n_types, h->d_cnt, h->d_ctot);
        k_exclusive_scan<<<1, 1024, 0, s>>>(nc, h->d_ctot, h->d_cstart);
        k_cm_rank<<<nb, 256, 0, s>>>(N, nc, h->d_key, h->d_sidx, h->d_start, h->d_cnt, h->d_cstart, h->d_cm, h->d_cmi);
        h->launches += 3;
    }
    h->launches += 4;
    int rc = qnep_launch_prep(h, pos, true, s);
    if (rc) return rc;
    const int nb2 = (int)((N + 127) / 128);
    k_build_lists<<<nb2, 128, 0, s>>>(N, h->model.n_types, h->geo, h->d_xyzt, h->d_cellc, h->d_start, h->capR,
                                     h->d_nlR, h->d_nnR, h->d_nnR0, h->d_nlRend, h->d_flags);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}

// out[0..5] = max / mean of the skin list, of the live radial list and of the live angular list (last call)
int qnep_launch_list_stats(qnep_handle* h, double out[6], cudaStream_t s)
{
    const int64_t N = h->N;
    const int nb = (int)((N + 255) / 256);
    struct Acc { unsigned long long sum[3]; int mx[3]; int pad; };
    Acc* d = nullptr;
    QNEP_CUDA_OK(h, cudaMalloc(&d, sizeof(Acc)));
    QNEP_CUDA_OK(h, cudaMemsetAsync(d, 0, sizeof(Acc), s));
    const int* arrays[3] = {h->d_nnR0, h->d_nlvR, h->d_nlvA};
    for (int a = 0; a < 3; ++a) k_count_stats<<<nb, 256, 0, s>>>(N, arrays[a], &d->mx[a], &d->sum[a]);
    h->launches += 3;
    Acc r;
    cudaError_t e = cudaMemcpyAsync(&r, d, sizeof(Acc), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(d);
    QNEP_CUDA_OK(h, e);
    for (int a = 0; a < 3; ++a) { out[2 * a] = r.mx[a]; out[2 * a + 1] = (double)r.sum[a] / (double)N; }
    return QNEP_OK;
}
