// pppm_sweep.cu -- step a7P-1 (charge assignment, Eq. 35) of SURVEY.md 8(a) on a shared-memory stencil tile,
// without atomics.
//
// Atoms are kept in MESH-BIN order (neighbor.cu, k_mbin_key): bins of MBX x MBY x MBZ = 4 x 8 x 8 mesh points, numbered
// column by column.  A block owns one (y, z) column of bins and SWEEPS it along x: a ring of SRING = 12 x-planes of the
// column's tile (TY = 14 rows y, TZ = 16 points z: the 8 x 8 bin cross-section plus the stencil halo of 2 and the drift
// margin of 1 mesh point the atoms may have moved since they were binned) lives in shared memory.
//
// k_spread_sweep: one warp per block.  The warp deposits ONE atom at a time: lane (b, c) of 25 adds
// q wx[a] wy[b] wz[c] to the five planes a -- all addresses of one atom are distinct, so plain ld/st.shared
// read-modify-write needs no atomic (shared-memory fp32 atomics are a CAS loop on sm_100a; the per-atom global
// reductions of the per-atom kernel are bound by the 1.3 cycles per lane the SM needs to issue a reduction).  The four
// planes that no later atom of the sweep can touch are moved to a dense staging box and added to the mesh with ONE
// cp.reduce.async.bulk.tensor (TMA reduction, UTMAREDG in SASS; a box that crosses the periodic boundary goes row by
// row through cp.reduce.async.bulk, UBLKRED, instead): the mesh receives one reduction per TILE point instead of 125
// per atom.
//
// The kernel needs the drift since the last neighbour build to stay within one mesh spacing (skin / 2 <= h_mesh),
// which qnep_sweep_usable() checks; otherwise, and for small systems (too few columns to fill 148 SMs), the per-atom
// kernel of pppm.cu runs.  An atom that moved further than skin / 2 adds nothing here; k_prep has flagged it
// (QNEP_ERR_SKIN_VIOLATED), so the result of such a step is discarded anyway.
//
// Back-interpolation (a7P-5) stays with the per-atom kernel of pppm.cu: a sweep version of it (TMA box loads of the
// float4 field planes into a 20-plane ring, eight lanes per atom reading the stencil from shared memory) was built and
// measured at 0.34 ms against 0.21 ms (profiles/r02_pppm_sweep.md): one warp instruction serves only four atoms there,
// and the 16 atoms of a step cannot amortise the per-step barrier / request / prefetch code.
#include "qnep_internal.cuh"

#include <algorithm>

#include "pppm_common.cuh"

#include <cmath>

namespace {

constexpr int MBX = QNEP_MB_X, MBY = QNEP_MB_Y, MBZ = QNEP_MB_Z;
constexpr int TY = MBY + 6;          // tile rows: y in [8 by - 3, 8 by + 11)
constexpr int TZ = MBZ + 8;          // tile points along z: [8 bz - 4, 8 bz + 12), 16-byte aligned at both ends
constexpr int SPZ = 19;              // spread: row pitch in floats: the banks 19 b + c of the 25 lanes (b, c) are all different
static_assert(MBX == 4 && MBY == 8 && MBZ == 8, "the window arithmetic below assumes 4 x 8 x 8 bins");

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bulk_red_add_f32(float* dst, const void* src, unsigned bytes)
{
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(NPENDING) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ int wrap(int v, int n) { v %= n; return v < 0 ? v + n : v; }

// offset of the nearest mesh point i0 (0 .. n-1) from the lowest one a bin admits (larger than the bin allows: the atom
// left its drift margin)
__device__ __forceinline__ int rel_index(int i0, int lo, int n)
{
    int v = i0 - lo;
    if (v < 0) v += n;
    if (v >= n) v -= n;
    return v;
}

struct SweepGeom {
    int n0, n1, n2;      // mesh
    int nbx, nbz;        // bins along x, z
    int segb, nseg;      // x bins per block (segment), segments per column
};

// the z run of a tile row in the mesh: one piece, or two when the column touches the periodic boundary
struct ZRun { int z[2], col[2], len[2], pieces; };
__device__ __forceinline__ ZRun z_run(int bz, int n2)
{
    ZRun r;
    const int zlo = MBZ * bz - 4;
    if (zlo < 0) { r.pieces = 2; r.z[0] = n2 + zlo; r.col[0] = 0; r.len[0] = -zlo; r.z[1] = 0; r.col[1] = -zlo; r.len[1] = TZ + zlo; }
    else if (zlo + TZ > n2) { r.pieces = 2; r.z[0] = zlo; r.col[0] = 0; r.len[0] = n2 - zlo; r.z[1] = 0; r.col[1] = n2 - zlo; r.len[1] = TZ - (n2 - zlo); }
    else { r.pieces = 1; r.z[0] = zlo; r.col[0] = 0; r.len[0] = TZ; r.z[1] = 0; r.col[1] = 0; r.len[1] = 0; }
    return r;
}

// ---- a7P-1: charge assignment ------------------------------------------------------------------------------
// Local plane index l = P - (4 b0 - 3) for the (unwrapped) mesh plane P; step s = b - b0 works on the window
// l in [4 s, 4 s + 10); ring slot = l mod SRING.  After step s the planes l < 4 s + 4 are final: they are copied to a
// staging box, zeroed in the ring (their slots are the next planes to enter the window) and reduced into the mesh.
constexpr int SRING = 12;
constexpr int AREC = 20;             // words of a prepared atom record (below)

__device__ __forceinline__ void tensor_red_add_3d(const CUtensorMap* tm, const void* src, int c0, int c1, int c2)
{
    asm volatile("cp.reduce.async.bulk.tensor.3d.global.shared::cta.add.tile.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tm), "r"(c0), "r"(c1),
                 "r"(c2), "r"(smem_u32(src))
                 : "memory");
}
// One warp per block (measured on config 4: 0.19 ms; with two warps, warp w depositing the planes whose ring slot has
// parity w, the kernel executes 1.5 x the instructions and takes 0.21 ms; the code below supports both).
constexpr int SP_THREADS = 32;
constexpr int SP_CHUNK = SP_THREADS; // atoms prepared at a time

__global__ void __launch_bounds__(SP_THREADS)
k_spread_sweep(const __grid_constant__ CUtensorMap tm_mesh, SweepGeom G, const int* __restrict__ mbstart,
               const float4* __restrict__ mfrac, const int2* __restrict__ qcm, float* __restrict__ mesh)
{
    __shared__ __align__(128) float stage[MBX * TY * TZ];         // dense box [4][14][16] for the TMA reduction
    __shared__ __align__(16) float ring[SRING * TY * SPZ];
    // prepared atoms of a chunk, one record per atom:
    //   words 0..3: ring offsets (BYTES) of the stencil origin in planes a = 0..3; bit 0 of word 0: parity of the slot of plane 0
    //   words 4..7: q wx[0..3];  word 8: offset in plane 4;  word 9: q wx[4];  words 10..14: wy;  words 15..19: wz
    //   (an atom that left its drift margin gets q = 0 and the offsets of the tile origin: it adds nothing)
    __shared__ __align__(16) float s_atom[SP_CHUNK * AREC];
    __shared__ int s_start[34];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int col = blockIdx.x / G.nseg, seg = blockIdx.x - col * G.nseg;
    const int by = col / G.nbz, bz = col - by * G.nbz;
    const int b0 = seg * G.segb, b1 = min(G.nbx, b0 + G.segb);
    const int nsteps = b1 - b0;
    const int kb0 = col * G.nbx + b0;
    if (tid <= nsteps) s_start[tid] = mbstart[kb0 + tid];        // first rank of every bin of the segment (segb <= 31)
    __syncthreads();
    const int q_begin = s_start[0], q_end = s_start[nsteps];
    if (q_begin == q_end) return;          // an empty stretch of the column (vacuum): nothing to add
    for (int i = tid; i < SRING * TY * SPZ / 4; i += SP_THREADS) reinterpret_cast<float4*>(ring)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    const int bb = lane / 5, cc = lane - 5 * bb;          // lanes 0..24: stencil row b, column c
    char* const ring_lane = reinterpret_cast<char*>(ring + bb * SPZ + cc);
    const ZRun zr = z_run(bz, G.n2);
    const int ylo = MBY * by - 3;
    const bool yz_inside = ylo >= 0 && ylo + TY <= G.n1 && zr.pieces == 1;
    int x0 = wrap(MBX * b0 - 3, G.n0);     // mesh plane of the next group of four planes to flush
    int fslot = 0;                         // its ring slot

    auto flush = [&]() {
        // planes [fslot, fslot + 4) of the ring (slots never wrap inside a group: SRING is a multiple of 4) are final
        bulk_wait_read<0>();               // the reduction of the previous flush (a whole step ago) is done with the box
        __syncthreads();                   // ... and every deposit of this step has been made
        // (the odd row pitch of the ring rules out vector accesses: thread -> column tid & 15 of the rows r, r + 2, ...)
#pragma unroll
        for (int pl = 0; pl < MBX; ++pl) {
#pragma unroll
            for (int r = 0; r < TY; r += SP_THREADS / 16) {
                const int row = r + (tid >> 4);
                if (row < TY) {
                    float* src = ring + ((fslot + pl) * TY + row) * SPZ + (tid & 15);
                    stage[(pl * TY + row) * TZ + (tid & 15)] = *src;
                    *src = 0.f;
                }
            }
        }
        fence_proxy_async();               // the box was written through the generic proxy
        __syncthreads();
        if (yz_inside && x0 + MBX <= G.n0) {
            if (tid == 0) tensor_red_add_3d(&tm_mesh, stage, zr.z[0], ylo, x0);
        } else {
            // the box crosses the periodic boundary (the TMA unit drops what lies beyond the END of an axis, but a
            // negative start coordinate of a store is an illegal instruction): one bulk reduction per row piece
            for (int i = tid; i < MBX * TY; i += SP_THREADS) {
                const int pl = i / TY, row = i - pl * TY;
                const int gx = x0 + pl >= G.n0 ? x0 + pl - G.n0 : x0 + pl;
                int gy = ylo + row;
                gy = gy < 0 ? gy + G.n1 : (gy >= G.n1 ? gy - G.n1 : gy);
                const float* src = stage + i * TZ;
                float* dst = mesh + ((int64_t)gx * G.n1 + gy) * G.n2;
                bulk_red_add_f32(dst + zr.z[0], src + zr.col[0], zr.len[0] * 4);
                if (zr.pieces == 2) bulk_red_add_f32(dst + zr.z[1], src + zr.col[1], zr.len[1] * 4);
            }
        }
        bulk_commit();
        x0 = x0 + MBX >= G.n0 ? x0 + MBX - G.n0 : x0 + MBX;
        fslot = fslot + MBX == SRING ? 0 : fslot + MBX;
    };

    // atom data of the next chunk, loaded one chunk ahead
    float4 fr = make_float4(0.f, 0.f, 0.f, 0.f);
    float qv = 0.f;
    auto load_chunk = [&](int qs) {
        const int qq = qs + tid;
        if (qq < q_end) { fr = mfrac[qq]; qv = __int_as_float(qcm[qq].y); }
    };
    load_chunk(q_begin);
    int wslot = 0;                         // ring slot of the first plane of the window of step s: (4 s) mod SRING

    for (int s = 0; s < nsteps; ++s) {
        const int b = b0 + s;
        const int qs_bin = s_start[s], qe_bin = s_start[s + 1];
        for (int qs = qs_bin; qs < qe_bin; qs += SP_CHUNK) {
            const int cnt = min(SP_CHUNK, qe_bin - qs);
            // thread t prepares atom t of the chunk
            if (tid < cnt) {
                float wx[5], wy[5], wz[5];
                bspline5(fr.x, wx); bspline5(fr.y, wy); bspline5(fr.z, wz);
                const int pk = __float_as_int(fr.w);
                int rx = rel_index(pk & 1023, MBX * b - 1, G.n0);
                int ry = rel_index((pk >> 10) & 1023, MBY * by - 1, G.n1);
                int rz = rel_index((pk >> 20) & 1023, MBZ * bz - 1, G.n2);
                const bool ok = rx <= MBX + 1 && ry <= MBY + 1 && rz <= MBZ + 1;
                const float qa = ok ? qv : 0.f;
                if (!ok) { rx = 0; ry = 0; rz = 0; }
                int off[5];
                int slot = wslot + rx;
                slot = slot >= SRING ? slot - SRING : slot;
                const int par = slot & 1;
                const int inplane = ry * SPZ + rz + 1;
#pragma unroll
                for (int a = 0; a < 5; ++a) {
                    off[a] = 4 * (slot * (TY * SPZ) + inplane);
                    slot = slot + 1 == SRING ? 0 : slot + 1;
                }
                float* rec = s_atom + tid * AREC;
                *reinterpret_cast<int4*>(rec) = make_int4(off[0] | par, off[1], off[2], off[3]);
                *reinterpret_cast<float4*>(rec + 4) = make_float4(qa * wx[0], qa * wx[1], qa * wx[2], qa * wx[3]);
                *reinterpret_cast<float4*>(rec + 8) = make_float4(__int_as_float(off[4]), qa * wx[4], wy[0], wy[1]);
                *reinterpret_cast<float4*>(rec + 12) = make_float4(wy[2], wy[3], wy[4], wz[0]);
                *reinterpret_cast<float4*>(rec + 16) = make_float4(wz[1], wz[2], wz[3], wz[4]);
            }
            __syncthreads();
            load_chunk(qs + cnt);          // the registers are free: request the next chunk (this bin's or a later one's)
            // both warps walk the atoms; warp w adds the planes whose ring slot has parity w (plane-disjoint: no race
            // between the warps; inside a warp one atom at a time).  The record of atom t + 1 is fetched while atom t is added.
            const float* rec = s_atom;
            int4 no = *reinterpret_cast<const int4*>(rec);
            float4 nw = *reinterpret_cast<const float4*>(rec + 4);
            float2 n8 = *reinterpret_cast<const float2*>(rec + 8);
            float nwy = rec[10 + bb], nwz = rec[15 + cc];
            for (int t = 0; t < cnt; ++t) {
                const int4 o = no;
                const float4 w = nw;
                const int o4 = __float_as_int(n8.x);
                const float w4 = n8.y;
                const float wyz = nwy * nwz;
                rec += (t + 1 < cnt) ? AREC : 0;
                no = *reinterpret_cast<const int4*>(rec);
                nw = *reinterpret_cast<const float4*>(rec + 4);
                n8 = *reinterpret_cast<const float2*>(rec + 8);
                nwy = rec[10 + bb]; nwz = rec[15 + cc];
                if (lane < 25) {
                    if (SP_THREADS == 32) {
                        float* const p0 = reinterpret_cast<float*>(ring_lane + (o.x & ~3));
                        float* const p1 = reinterpret_cast<float*>(ring_lane + o.y);
                        float* const p2 = reinterpret_cast<float*>(ring_lane + o.z);
                        float* const p3 = reinterpret_cast<float*>(ring_lane + o.w);
                        float* const p4 = reinterpret_cast<float*>(ring_lane + o4);
                        const float v0 = *p0, v1 = *p1, v2 = *p2, v3 = *p3, v4 = *p4;
                        *p0 = fmaf(w.x, wyz, v0);
                        *p1 = fmaf(w.y, wyz, v1);
                        *p2 = fmaf(w.z, wyz, v2);
                        *p3 = fmaf(w.w, wyz, v3);
                        *p4 = fmaf(w4, wyz, v4);
                    } else if (((o.x ^ warp) & 1) == 0) {
                        float* const p0 = reinterpret_cast<float*>(ring_lane + (o.x & ~3));
                        float* const p2 = reinterpret_cast<float*>(ring_lane + o.z);
                        float* const p4 = reinterpret_cast<float*>(ring_lane + o4);
                        const float v0 = *p0, v2 = *p2, v4 = *p4;
                        *p0 = fmaf(w.x, wyz, v0);
                        *p2 = fmaf(w.z, wyz, v2);
                        *p4 = fmaf(w4, wyz, v4);
                    } else {
                        float* const p1 = reinterpret_cast<float*>(ring_lane + o.y);
                        float* const p3 = reinterpret_cast<float*>(ring_lane + o.w);
                        const float v1 = *p1, v3 = *p3;
                        *p1 = fmaf(w.y, wyz, v1);
                        *p3 = fmaf(w.w, wyz, v3);
                    }
                }
                __syncwarp();
            }
            if (qs + SP_CHUNK < qe_bin) __syncthreads();      // the records are rewritten for the next chunk of this bin
        }
        flush();
        wslot = wslot + MBX == SRING ? 0 : wslot + MBX;
    }
    // the tail of the last window: planes 4 n .. 4 n + 5 (the two planes after them are zero in the ring)
    flush();
    flush();
    bulk_wait_read<0>();                   // shared memory must outlive the reads of the bulk operations
}

SweepGeom sweep_geom(const qnep_handle* h)
{
    SweepGeom G;
    G.n0 = h->geo.grid[0]; G.n1 = h->geo.grid[1]; G.n2 = h->geo.grid[2];
    G.nbx = h->nmb[0]; G.nbz = h->nmb[2];
    // segments of at most 16 bins (64 planes): the tail of 6 planes a segment flushes / the 8 it loads first are amortised
    G.nseg = (G.nbx + 15) / 16;
    G.segb = (G.nbx + G.nseg - 1) / G.nseg;
    return G;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

}  // namespace

// TMA descriptors of the charge mesh and of the field mesh (called by qnep_setup_pppm after the meshes are allocated)
int qnep_setup_sweep(qnep_handle* h)
{
    h->tm_ok = false;
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
            cudaGetLastError();
            return QNEP_OK;              // no TMA descriptors: the per-atom kernels run
        }
        encode = (EncodeTiledFn)fn;
    }
    const cuuint64_t n0 = h->es.grid[0], n1 = h->es.grid[1], n2 = h->es.grid[2];
    const cuuint32_t estr[3] = {1, 1, 1};
    {
        const cuuint64_t dims[3] = {n2, n1, n0};
        const cuuint64_t strides[2] = {n2 * sizeof(float), n1 * n2 * sizeof(float)};
        const cuuint32_t box[3] = {(cuuint32_t)TZ, (cuuint32_t)TY, (cuuint32_t)MBX};
        if (encode(&h->tm_mesh, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, h->d_mesh, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return QNEP_OK;
    }
    h->tm_ok = true;
    return QNEP_OK;
}

// the sweep kernels apply when the drift margin of one mesh point covers skin / 2 (header comment); automatic mode also
// asks for enough atoms to fill the GPU with columns
bool qnep_sweep_usable(const qnep_handle* h)
{
    if (h->es.method != 2 || h->nmbins == 0 || h->pppm_kernels == 1 || !h->tm_ok) return false;
    for (int a = 0; a < 3; ++a) {
        // a displacement of skin / 2 changes the mesh coordinate along a by at most skin / 2 * |b*_a| * grid_a (any cell)
        const double* hi = h->geo.hinv;
        const double bnorm = std::sqrt(hi[a] * hi[a] + hi[3 + a] * hi[3 + a] + hi[6 + a] * hi[6 + a]);
        if (0.5 * h->skin * bnorm * h->geo.grid[a] > 1.0) return false;
    }
    // automatic: the kernel runs one warp per column segment, so it needs thousands of columns to fill the GPU (1024 x 4
    // at 256^3: 0.19 ms against 0.23 ms; at 128^3 and 64^3 the per-atom kernel is faster: 0.22 / 0.29 ms and 0.05 / 0.17 ms
    // per reciprocal stage on configs 3 and 2)
    return h->pppm_kernels == 2 || (h->N >= QNEP_SWEEP_MIN_ATOMS && h->nmb[1] * h->nmb[2] >= 1024);
}

int qnep_launch_spread_sweep(qnep_handle* h, cudaStream_t s)
{
    const SweepGeom G = sweep_geom(h);
    const unsigned nblocks = (unsigned)(h->nmb[1] * h->nmb[2] * G.nseg);
    QNEP_CUDA_OK(h, cudaMemsetAsync(h->d_mesh, 0, sizeof(float) * h->ngrid, s));
    k_spread_sweep<<<nblocks, SP_THREADS, 0, s>>>(h->tm_mesh, G, h->d_mbstart, h->d_mfrac, h->d_qcm, h->d_mesh);
    h->launches += 1;
    QNEP_CUDA_OK(h, cudaGetLastError());
    return QNEP_OK;
}
