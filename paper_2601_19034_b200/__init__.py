"""paper_2601_19034_b200 -- thin Python binding of the C-ABI library ``libqnep_b200.so``
(include/qnep.h): the B200-native qNEP force evaluation of arXiv 2601.19034.

Argument marshalling only: every step of the path runs in the CUDA kernels of ``csrc/``.
PyTorch supplies device memory and streams.  There is NO CPU fallback: importing works
anywhere (so the C ABI can be inspected), but creating a handle without the built library
or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libqnep_b200.so")

QNEP_OK = 0
QNEP_ERR_INVALID_ARG = -1
QNEP_ERR_UNSUPPORTED = -2
QNEP_ERR_NEIGHBOR_OVERFLOW = -3
QNEP_ERR_SKIN_VIOLATED = -4
QNEP_ERR_CUDA = -5
QNEP_ERR_OOM = -6
ERROR_NAMES = {0: "OK", -1: "INVALID_ARG", -2: "UNSUPPORTED", -3: "NEIGHBOR_OVERFLOW", -4: "SKIN_VIOLATED",
               -5: "CUDA", -6: "OOM"}

WANT_ENERGY, WANT_FORCES, WANT_VIRIAL, WANT_CHARGES, WANT_BEC, WANT_ATOM_VIRIAL = 1, 2, 4, 8, 16, 32
WANT_ALL = WANT_ENERGY | WANT_FORCES | WANT_VIRIAL | WANT_CHARGES

TIMING_NAMES = ["neighbor", "prep", "desc_radial", "desc_angular", "nn", "realspace", "reciprocal",
                "force_angular", "force_radial", "bec", "total"]
DBG_DESCRIPTORS, DBG_SITE_ENERGY, DBG_Q_RAW, DBG_PHI, DBG_FP, DBG_MESH_RHO, DBG_F_STATIC, DBG_ENERGY_PARTS = range(8)

# every symbol include/qnep.h declares
ABI_SYMBOLS = ["qnep_create", "qnep_set_electrostatics", "qnep_set_neighbor_policy", "qnep_set_neighbor_capacity",
               "qnep_compute", "qnep_compute_atom_virial", "qnep_compute_host", "qnep_md_run", "qnep_md_set_outputs", "qnep_md_reset", "qnep_set_md_graphs", "qnep_set_pppm_kernels", "qnep_check", "qnep_get_timings",
               "qnep_profile_reset", "qnep_profile_sum", "qnep_kernel_launches", "qnep_response", "qnep_neighbor_stats",
               "qnep_fma_peak", "qnep_set_zbl", "qnep_set_nn_kernel",
               "qnep_debug_copy", "qnep_neutralise_noalloc", "qnep_abi_version", "qnep_destroy", "qnep_last_error"]
ABI_VERSION = 3                      # QNEP_ABI_VERSION of the include/qnep.h these ctypes mirrors were written against
NOALLOC_MAX_ATOMS = 4194304          # QNEP_NOALLOC_MAX_ATOMS of include/qnep.h


class qnep_model_desc(C.Structure):
    _fields_ = [("n_types", C.c_int32), ("n_max_r", C.c_int32), ("n_max_a", C.c_int32), ("l_max", C.c_int32),
                ("basis_r", C.c_int32), ("basis_a", C.c_int32), ("n_neurons", C.c_int32),
                ("rc_r", C.c_double), ("rc_a", C.c_double), ("mode", C.c_int32),
                ("sqrt_eps_inf", C.c_double), ("q_total", C.c_double), ("l_max_4b", C.c_int32), ("l_max_5b", C.c_int32)]


class qnep_es_desc(C.Structure):
    _fields_ = [("method", C.c_int32), ("alpha", C.c_double), ("ewald_nmax2", C.c_int32),
                ("grid", C.c_int32 * 3), ("order", C.c_int32)]


class QnepError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"QNEP_ERR_{ERROR_NAMES.get(code, code)}: {message}")
        self.code = code


_lib = None


def load_library():
    """dlopen libqnep_b200.so; raises (loudly) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2601_19034_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.qnep_abi_version.restype = C.c_int
    lib.qnep_abi_version.argtypes = []
    if lib.qnep_abi_version() != ABI_VERSION:
        raise ImportError(f"{LIB_PATH} was built from a header of ABI version {lib.qnep_abi_version()}, this binding mirrors "
                          f"version {ABI_VERSION}: rebuild with `python -m paper_2601_19034_b200.build --force`")
    vp, i64, i32, u32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_uint32, C.c_double
    lib.qnep_create.restype = C.c_int
    lib.qnep_create.argtypes = [C.POINTER(qnep_model_desc), vp, C.c_size_t, C.POINTER(qnep_es_desc), C.POINTER(vp)]
    lib.qnep_set_electrostatics.restype = C.c_int
    lib.qnep_set_electrostatics.argtypes = [vp, C.POINTER(qnep_es_desc)]
    lib.qnep_set_neighbor_policy.restype = C.c_int
    lib.qnep_set_neighbor_policy.argtypes = [vp, dbl, i32]
    lib.qnep_set_neighbor_capacity.restype = C.c_int
    lib.qnep_set_neighbor_capacity.argtypes = [vp, i32, i32]
    for name in ("qnep_compute", "qnep_compute_host"):
        f = getattr(lib, name)
        f.restype = C.c_int
        f.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), u32, vp, vp, vp, vp, vp, vp]
    lib.qnep_compute_atom_virial.restype = C.c_int
    lib.qnep_compute_atom_virial.argtypes = [vp, i64, vp, vp, C.POINTER(dbl), u32, vp, vp, vp, vp, vp, vp]
    lib.qnep_md_run.restype = C.c_int
    lib.qnep_md_run.argtypes = [vp, i64, vp, vp, vp, C.POINTER(dbl), C.POINTER(dbl), dbl, i32, vp, vp]
    lib.qnep_check.restype = C.c_int
    lib.qnep_md_set_outputs.restype = C.c_int
    lib.qnep_md_set_outputs.argtypes = [vp, u32, vp, vp]
    lib.qnep_md_reset.restype = C.c_int
    lib.qnep_md_reset.argtypes = [vp]
    lib.qnep_set_md_graphs.restype = C.c_int
    lib.qnep_set_md_graphs.argtypes = [vp, i32]
    lib.qnep_check.argtypes = [vp]
    lib.qnep_set_pppm_kernels.restype = C.c_int
    lib.qnep_set_pppm_kernels.argtypes = [vp, i32]
    lib.qnep_get_timings.restype = C.c_int
    lib.qnep_get_timings.argtypes = [vp, C.POINTER(C.c_float), i32]
    lib.qnep_profile_reset.restype = C.c_int
    lib.qnep_profile_reset.argtypes = [vp]
    lib.qnep_profile_sum.restype = C.c_int
    lib.qnep_profile_sum.argtypes = [vp, C.POINTER(C.c_float), i32, C.POINTER(i64)]
    lib.qnep_kernel_launches.restype = i64
    lib.qnep_kernel_launches.argtypes = [vp]
    lib.qnep_response.restype = C.c_int
    lib.qnep_response.argtypes = [vp, i64, vp, C.POINTER(dbl), vp, vp, vp, vp]
    lib.qnep_neighbor_stats.restype = C.c_int
    lib.qnep_neighbor_stats.argtypes = [vp, C.POINTER(dbl)]
    lib.qnep_set_nn_kernel.restype = C.c_int
    lib.qnep_set_nn_kernel.argtypes = [vp, i32]
    lib.qnep_set_zbl.restype = C.c_int
    lib.qnep_set_zbl.argtypes = [vp, i32, dbl, dbl, C.POINTER(dbl)]
    lib.qnep_fma_peak.restype = C.c_int
    lib.qnep_fma_peak.argtypes = [C.POINTER(dbl), vp]
    lib.qnep_debug_copy.restype = C.c_int
    lib.qnep_debug_copy.argtypes = [vp, i32, vp, i64]
    lib.qnep_neutralise_noalloc.restype = C.c_int
    lib.qnep_neutralise_noalloc.argtypes = [i64, vp, dbl, vp, vp, C.c_char_p, C.c_size_t]
    lib.qnep_destroy.restype = None
    lib.qnep_destroy.argtypes = [vp]
    lib.qnep_last_error.restype = C.c_char_p
    lib.qnep_last_error.argtypes = [vp]
    _lib = lib
    return lib


def _model_struct(m) -> qnep_model_desc:
    return qnep_model_desc(m.n_types, m.n_max_r, m.n_max_a, m.l_max, m.basis_r, m.basis_a, m.n_neurons,
                           m.rc_r, m.rc_a, m.mode, m.sqrt_eps_inf, m.q_total, getattr(m, "l_max_4b", 0), getattr(m, "l_max_5b", 0))


def _es_struct(e) -> qnep_es_desc:
    return qnep_es_desc(e.method, e.alpha, e.ewald_nmax2, (C.c_int32 * 3)(*e.grid), e.order)


def _box(box):
    b = np.ascontiguousarray(np.asarray(box, dtype=np.float64).ravel())
    assert b.shape[0] == 9
    return (C.c_double * 9)(*b)


class QNEP:
    """A handle of the C library.  Methods carry the names of the C entry points (qnep_ prefix dropped)."""

    def __init__(self, model, params, es):
        self._lib = load_library()
        p = np.ascontiguousarray(params, dtype=np.float32)
        self._h = C.c_void_p()
        self.model = model
        m, e = _model_struct(model), _es_struct(es)
        rc = self._lib.qnep_create(C.byref(m), p.ctypes.data_as(C.c_void_p), p.shape[0], C.byref(e), C.byref(self._h))
        if rc != QNEP_OK:
            raise QnepError(rc, self._lib.qnep_last_error(None).decode())

    # -- plumbing ---------------------------------------------------------------------------
    def _ok(self, rc):
        if rc != QNEP_OK:
            raise QnepError(rc, self._lib.qnep_last_error(self._h).decode())

    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.qnep_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @staticmethod
    def _stream(stream):
        import torch
        s = torch.cuda.current_stream() if stream is None else stream
        return C.c_void_p(s.cuda_stream)

    # -- entry points -----------------------------------------------------------------------
    def set_electrostatics(self, es):
        e = _es_struct(es)
        self._ok(self._lib.qnep_set_electrostatics(self._h, C.byref(e)))

    def set_neighbor_policy(self, skin: float, rebuild_every: int):
        self._ok(self._lib.qnep_set_neighbor_policy(self._h, float(skin), int(rebuild_every)))

    def set_neighbor_capacity(self, cap_radial: int, cap_angular: int):
        self._ok(self._lib.qnep_set_neighbor_capacity(self._h, int(cap_radial), int(cap_angular)))

    def compute(self, pos, types, box, want=WANT_ALL, out=None, stream=None, check=True):
        """pos: cuda float64 [3][N]; types: cuda int32 [N]; box: 9 floats (host).  Returns dict of cuda tensors."""
        import torch
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous() and pos.shape[0] == 3
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        n = pos.shape[1]
        dev = pos.device
        if out is None:
            out = {}
        def buf(key, flag, shape):
            if not (want & flag):
                return None
            if key not in out:
                out[key] = torch.empty(shape, dtype=torch.float64, device=dev)
            return out[key]
        e = buf("energy", WANT_ENERGY, (1,))
        f = buf("forces", WANT_FORCES, (3, n))
        w = buf("virial", WANT_VIRIAL, (9,))
        q = buf("charges", WANT_CHARGES, (n,))
        z = buf("bec", WANT_BEC, (9, n))
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        rc = self._lib.qnep_compute(self._h, n, ptr(pos), ptr(types), _box(box), want, ptr(e), ptr(f), ptr(w), ptr(q),
                                    ptr(z), self._stream(stream))
        self._ok(rc)
        if check:
            self.check()
        return out

    def compute_atom_virial(self, pos, types, box, want=WANT_ALL, stream=None):
        """qnep_compute_atom_virial: the outputs of compute() plus "virial_atom" [9][N] (Eq. 12, 20, 39)."""
        import torch
        assert pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous() and pos.shape[0] == 3
        assert types.is_cuda and types.dtype == torch.int32 and types.is_contiguous()
        n = pos.shape[1]
        out = {"virial_atom": torch.empty((9, n), dtype=torch.float64, device=pos.device)}
        def buf(key, flag, shape):
            if not (want & flag):
                return None
            out[key] = torch.empty(shape, dtype=torch.float64, device=pos.device)
            return out[key]
        e = buf("energy", WANT_ENERGY, (1,))
        f = buf("forces", WANT_FORCES, (3, n))
        w = buf("virial", WANT_VIRIAL, (9,))
        q = buf("charges", WANT_CHARGES, (n,))
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        rc = self._lib.qnep_compute_atom_virial(self._h, n, ptr(pos), ptr(types), _box(box), want, ptr(e), ptr(f), ptr(w),
                                                ptr(q), ptr(out["virial_atom"]), self._stream(stream))
        self._ok(rc)
        self.check()
        return out

    def compute_host(self, pos, types, box, want=WANT_ALL, stream=None):
        """Host numpy buffers in, host numpy buffers out (copies inside the call)."""
        pos = np.ascontiguousarray(pos, dtype=np.float64)
        types = np.ascontiguousarray(types, dtype=np.int32)
        n = pos.shape[1]
        out = {}
        def buf(key, flag, shape):
            if want & flag:
                out[key] = np.empty(shape, dtype=np.float64)
                return out[key].ctypes.data_as(C.c_void_p)
            return None
        e = buf("energy", WANT_ENERGY, (1,))
        f = buf("forces", WANT_FORCES, (3, n))
        w = buf("virial", WANT_VIRIAL, (9,))
        q = buf("charges", WANT_CHARGES, (n,))
        z = buf("bec", WANT_BEC, (9, n))
        rc = self._lib.qnep_compute_host(self._h, n, pos.ctypes.data_as(C.c_void_p), types.ctypes.data_as(C.c_void_p),
                                         _box(box), want, e, f, w, q, z, self._stream(stream))
        self._ok(rc)
        return out

    def compute_host_raw(self, n, pos_ptr, types_ptr, box9, want, e_ptr, f_ptr, w_ptr, q_ptr, z_ptr, stream=None):
        """qnep_compute_host with caller-managed (e.g. pinned) host pointers given as integers."""
        vp = lambda x: C.c_void_p(x) if x else None
        rc = self._lib.qnep_compute_host(self._h, n, vp(pos_ptr), vp(types_ptr), box9, want, vp(e_ptr), vp(f_ptr),
                                         vp(w_ptr), vp(q_ptr), vp(z_ptr), self._stream(stream))
        self._ok(rc)

    def md_run(self, pos, vel, types, box, masses, dt, n_steps, stream=None):
        import torch
        assert pos.is_cuda and vel.is_cuda and pos.dtype == torch.float64 and vel.dtype == torch.float64
        n = pos.shape[1]
        energy = torch.zeros(2, dtype=torch.float64, device=pos.device)
        m = np.ascontiguousarray(masses, dtype=np.float64)
        rc = self._lib.qnep_md_run(self._h, n, C.c_void_p(pos.data_ptr()), C.c_void_p(vel.data_ptr()),
                                   C.c_void_p(types.data_ptr()), _box(box), m.ctypes.data_as(C.POINTER(C.c_double)),
                                   float(dt), int(n_steps), C.c_void_p(energy.data_ptr()), self._stream(stream))
        self._ok(rc)
        return energy

    def check(self):
        self._ok(self._lib.qnep_check(self._h))

    def get_timings(self) -> dict:
        ms = (C.c_float * len(TIMING_NAMES))()
        self._ok(self._lib.qnep_get_timings(self._h, ms, len(TIMING_NAMES)))
        return {k: float(v) for k, v in zip(TIMING_NAMES, ms)}

    def profile_reset(self):
        self._ok(self._lib.qnep_profile_reset(self._h))

    def profile_sum(self):
        """(dict of summed stage times in ms, number of evaluations summed)."""
        ms = (C.c_float * len(TIMING_NAMES))()
        n = C.c_int64(0)
        self._ok(self._lib.qnep_profile_sum(self._h, ms, len(TIMING_NAMES), C.byref(n)))
        return {k: float(v) for k, v in zip(TIMING_NAMES, ms)}, int(n.value)

    def kernel_launches(self) -> int:
        return int(self._lib.qnep_kernel_launches(self._h))

    def md_set_outputs(self, virial=None, charges=None):
        """Extra outputs of the steps of md_run: cuda float64 tensors virial [9] and / or charges [N] (kept alive by the
        caller), or neither to restore the default (energy and forces only)."""
        want = (WANT_VIRIAL if virial is not None else 0) | (WANT_CHARGES if charges is not None else 0)
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._ok(self._lib.qnep_md_set_outputs(self._h, want, ptr(virial), ptr(charges)))
        self._md_outputs = (virial, charges)

    def md_reset(self):
        """Positions / velocities were changed outside md_run: drop the kept forces, rebuild the lists next time."""
        self._ok(self._lib.qnep_md_reset(self._h))

    def set_md_graphs(self, mode: int):
        """0 never, 1 (default) for n_atoms <= 100000, 2 always: CUDA graphs for the steps of md_run."""
        self._ok(self._lib.qnep_set_md_graphs(self._h, int(mode)))

    def set_pppm_kernels(self, mode: int):
        """0 automatic, 1 one thread per atom, 2 shared-memory sweep kernel: PPPM charge assignment."""
        self._ok(self._lib.qnep_set_pppm_kernels(self._h, int(mode)))

    def set_nn_kernel(self, mode: int):
        """2 (default for the 25-descriptor model with n_neurons <= 128): tcgen05 tensor cores, 3xTF32 split; 1: mma.sync
        TF32, same split; 0: packed FP32 FMAs (the default otherwise).  UNSUPPORTED: modes 1, 2 with the 4-/5-body terms on,
        mode 2 with n_neurons > 128, mode 1 when n_types x n_neurons needs more than 200 KB of shared memory."""
        self._ok(self._lib.qnep_set_nn_kernel(self._h, int(mode)))

    def set_zbl(self, zbl):
        """zbl = (r_inner, r_outer, Z per species) switches the ZBL core on, None switches it off."""
        if zbl is None:
            self._ok(self._lib.qnep_set_zbl(self._h, 0, 0.0, 0.0, None))
        else:
            r1, r2, Z = zbl
            Z = (C.c_double * len(Z))(*[float(v) for v in Z])
            self._ok(self._lib.qnep_set_zbl(self._h, 1, float(r1), float(r2), Z))

    def response(self, bec, efield=None, vel=None, stream=None):
        """Eq. 29-30 from the BEC tensor [9][N] (cuda float64): returns (fext [3][N] or None, pdot [3] or None)."""
        import torch
        assert bec.is_cuda and bec.dtype == torch.float64 and bec.is_contiguous() and bec.shape[0] == 9
        n = bec.shape[1]
        fext = torch.empty((3, n), dtype=torch.float64, device=bec.device) if efield is not None else None
        pdot = torch.empty(3, dtype=torch.float64, device=bec.device) if vel is not None else None
        if vel is not None:
            assert vel.is_cuda and vel.dtype == torch.float64 and vel.is_contiguous() and tuple(vel.shape) == (3, n)
        e3 = (C.c_double * 3)(*[float(x) for x in efield]) if efield is not None else None
        ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
        self._ok(self._lib.qnep_response(self._h, n, ptr(bec), e3, ptr(vel), ptr(fext), ptr(pdot), self._stream(stream)))
        return fext, pdot

    def neighbor_stats(self) -> dict:
        out = (C.c_double * 6)()
        self._ok(self._lib.qnep_neighbor_stats(self._h, out))
        return dict(max_list=out[0], mean_list=out[1], max_radial=out[2], mean_radial=out[3],
                    max_angular=out[4], mean_angular=out[5])

    def debug_copy(self, which: int, shape):
        import torch
        t = torch.zeros(shape, dtype=torch.float64, device="cuda")
        self._ok(self._lib.qnep_debug_copy(self._h, which, C.c_void_p(t.data_ptr()), t.numel()))
        return t


def fma_peak(stream=None) -> float:
    """Measured FP32 FMA throughput of the current device, TFLOP/s (qnep_fma_peak)."""
    out = C.c_double(0.0)
    rc = load_library().qnep_fma_peak(C.byref(out), QNEP._stream(stream))
    if rc != QNEP_OK:
        raise QnepError(rc, "qnep_fma_peak failed")
    return float(out.value)


def neutralise_noalloc(q_raw, q_total: float, out=None, stream=None):
    """qnep_neutralise_noalloc: Eq. 33, ``out_i = q_raw_i + (q_total - sum q_raw) / N``, without a handle and without any
    device allocation inside the library -- for callers whose GPU memory is owned by someone else's pool, or who may not
    stall the device with cudaMalloc / cudaFree (see include/qnep.h).  q_raw: cuda float64 [N], N <= NOALLOC_MAX_ATOMS;
    out: cuda float64 [N] supplied by the caller (``out=q_raw`` works in place); only when it is None does this
    convenience wrapper -- not the library -- take one from torch.  All calls on a device share one built-in scratch array:
    do not let two of them run at the same time on different streams.  The first call on a device does a one-off set-up."""
    import torch
    assert q_raw.is_cuda and q_raw.dtype == torch.float64 and q_raw.is_contiguous() and q_raw.dim() == 1
    if out is None:
        out = torch.empty_like(q_raw)
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.shape == q_raw.shape
    msg = C.create_string_buffer(512)
    with torch.cuda.device(q_raw.device):
        rc = load_library().qnep_neutralise_noalloc(q_raw.shape[0], C.c_void_p(q_raw.data_ptr()), float(q_total),
                                                    C.c_void_p(out.data_ptr()), QNEP._stream(stream), msg, len(msg))
    if rc != QNEP_OK:
        raise QnepError(rc, msg.value.decode())
    return out


def from_workload(w) -> QNEP:
    """Handle for a qnep_inputs.Workload."""
    h = QNEP(w.model, w.params, w.es)
    if getattr(w, "zbl", None) is not None:
        h.set_zbl(w.zbl)
    return h
