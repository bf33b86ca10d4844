"""ctypes binding of the fp64 CPU oracle (oracle/qnep_oracle.c).

TEST INFRASTRUCTURE ONLY (see the header of qnep_oracle.c): imported by tests/,
by __graft_entry__.smoke() and by bench.py's cpu_baseline / --impl reference
legs.  The product package never imports this module.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qnep_oracle.c")
_LIB = os.path.join(_HERE, "libqnep_oracle.so")

K_COULOMB = 14.3996454784  # eV*A/e^2 (reading S9); repeated here only for the tests' closed forms


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99 + OpenMP).

    QNEP_ORACLE_SANITIZE=1 builds a second library with -fsanitize=address,undefined instead; run the
    CPU tests on it with  LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0."""
    if os.environ.get("QNEP_ORACLE_SANITIZE") == "1":
        lib_ = os.path.join(_HERE, "libqnep_oracle_san.so")
        if force or not os.path.exists(lib_) or os.path.getmtime(lib_) < os.path.getmtime(_SRC):
            cmd = ["gcc", "-O1", "-g", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-fsanitize=address,undefined",
                   "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-o", lib_, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
        return lib_
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Model(C.Structure):
    _fields_ = [("n_types", C.c_int32), ("n_max_r", C.c_int32), ("n_max_a", C.c_int32), ("l_max", C.c_int32),
                ("basis_r", C.c_int32), ("basis_a", C.c_int32), ("n_neurons", C.c_int32),
                ("rc_r", C.c_double), ("rc_a", C.c_double), ("mode", C.c_int32),
                ("sqrt_eps_inf", C.c_double), ("q_total", C.c_double), ("l_max_4b", C.c_int32), ("l_max_5b", C.c_int32)]


class _Es(C.Structure):
    _fields_ = [("method", C.c_int32), ("alpha", C.c_double), ("ewald_nmax2", C.c_int32),
                ("grid", C.c_int32 * 3), ("order", C.c_int32)]


class _Debug(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("D", "U_i", "q_raw", "phi", "Fp", "rho", "F_es")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_alias_denominator.restype = C.c_double
        _lib.orc_alias_denominator.argtypes = [C.c_double]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _model(m) -> _Model:
    return _Model(m.n_types, m.n_max_r, m.n_max_a, m.l_max, m.basis_r, m.basis_a, m.n_neurons,
                  m.rc_r, m.rc_a, m.mode, m.sqrt_eps_inf, m.q_total, getattr(m, "l_max_4b", 0), getattr(m, "l_max_5b", 0))


def _es(e) -> _Es:
    return _Es(e.method, e.alpha, e.ewald_nmax2, (C.c_int32 * 3)(*e.grid), e.order)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def neighbors(pos, box, rc, use_bins=False, cap=0):
    pos = _f64(pos)
    n = pos.shape[1]
    counts = np.zeros(n, dtype=np.int64)
    oj = np.full((n, max(cap, 1)), -1, dtype=np.int32)
    od = np.zeros((n, max(cap, 1), 4))
    rc_ = lib().orc_neighbors(C.c_int64(n), _p(pos), _p(_f64(box)), C.c_double(rc), C.c_int(int(use_bins)),
                              _p(counts), C.c_int64(cap), _p(oj), _p(od))
    assert rc_ == 0
    return counts, oj, od


def descriptors(model, params, pos, types, box, use_bins=False):
    pos = _f64(pos)
    n = pos.shape[1]
    D = np.zeros((n, model.n_desc))
    mm = _model(model)
    rc_ = lib().orc_descriptors(C.byref(mm), _p(_f64(params)), C.c_int64(n), _p(pos),
                                _p(np.ascontiguousarray(types, dtype=np.int32)), _p(_f64(box)),
                                C.c_int(int(use_bins)), _p(D))
    assert rc_ == 0, rc_
    return D


def electrostatics(pos, q, box, rc, mode, es, want_rho=False, want_atom_virial=False):
    """Fixed charges -> dict(U=[U^r, U^k, U^s], phi, F[3][N], W[3][3], rho, W_atom[9][N])."""
    pos = _f64(pos)
    n = pos.shape[1]
    U = np.zeros(3)
    phi = np.zeros(n)
    F = np.zeros((3, n))
    W = np.zeros(9)
    rho = np.zeros(tuple(es.grid)) if (want_rho and es.method == 2) else None
    ee = _es(es)
    Wat = np.zeros((9, n)) if want_atom_virial else None
    rc_ = lib().orc_electrostatics(C.c_int64(n), _p(pos), _p(_f64(q)), _p(_f64(box)), C.c_double(rc),
                                   C.c_int(mode), C.byref(ee), _p(U), _p(phi), _p(F), _p(W), _p(rho), _p(Wat))
    assert rc_ == 0, rc_
    return dict(U=U, phi=phi, F=F, W=W.reshape(3, 3), rho=rho, W_atom=Wat)


def compute(model, params, es, pos, types, box, use_bins=True, want_bec=False, debug=False, want_atom_virial=False, zbl=None):
    """The whole force evaluation.  Returns a dict of fp64 arrays.  zbl = (r_inner, r_outer, Z per species) switches the
    ZBL core on for this call (reading Z1)."""
    pos = _f64(pos)
    n = pos.shape[1]
    Dn = model.n_desc
    energy = np.zeros(6)
    forces = np.zeros((3, n))
    virial = np.zeros(9)
    charges = np.zeros(n)
    bec = np.zeros((9, n)) if want_bec else None
    wat = np.zeros((9, n)) if want_atom_virial else None
    out = {}
    dbg = None
    if debug:
        out["D"] = np.zeros((n, Dn))
        out["U_i"] = np.zeros(n)
        out["q_raw"] = np.zeros(n)
        out["phi"] = np.zeros(n)
        out["Fp"] = np.zeros((n, Dn))
        out["rho"] = np.zeros(tuple(es.grid)) if es.method == 2 else None
        out["F_es"] = np.zeros((3, n))
        dbg = _Debug(*[_p(out[k]) for k in ("D", "U_i", "q_raw", "phi", "Fp", "rho", "F_es")])
    mm, ee = _model(model), _es(es)
    set_zbl(zbl, model.n_types)
    try:
        rc_ = _call_compute(mm, params, ee, n, pos, types, box, use_bins, energy, forces, virial, charges, bec, dbg, wat)
    finally:
        set_zbl(None, model.n_types)
    if rc_ != 0:
        raise RuntimeError(f"orc_compute failed with code {rc_}")
    out.update(energy=energy[0], energy_parts=dict(nep=energy[1], r=energy[2], k=energy[3], s=energy[4], zbl=energy[5]),
               forces=forces, virial=virial.reshape(3, 3), charges=charges, bec=bec, virial_atom=wat)
    return out


def set_zbl(zbl, n_types):
    f = lib().orc_set_zbl
    f.restype = None
    if zbl is None:
        f(C.c_int(0), C.c_double(0.0), C.c_double(0.0), None, C.c_int(0))
    else:
        r1, r2, Z = zbl
        Z = _f64(np.asarray(Z, dtype=np.float64))
        assert len(Z) >= n_types
        f(C.c_int(1), C.c_double(r1), C.c_double(r2), _p(Z), C.c_int(n_types))


def zbl_pair(r, Zi, Zj, r1, r2):
    """(U_ZBL(r), dU_ZBL/dr) of one pair (reading Z1)."""
    u, du = C.c_double(0.0), C.c_double(0.0)
    f = lib().orc_zbl_pair
    f.restype = None
    f(C.c_double(r), C.c_double(Zi), C.c_double(Zj), C.c_double(r1), C.c_double(r2), C.byref(u), C.byref(du))
    return u.value, du.value


def _call_compute(mm, params, ee, n, pos, types, box, use_bins, energy, forces, virial, charges, bec, dbg, wat):
    return lib().orc_compute(C.byref(mm), _p(_f64(params)), C.byref(ee), C.c_int64(n), _p(pos),
                            _p(np.ascontiguousarray(types, dtype=np.int32)), _p(_f64(box)),
                            C.c_int(int(use_bins)), _p(energy), _p(forces), _p(virial), _p(charges), _p(bec),
                            C.byref(dbg) if dbg is not None else None, _p(wat))


def response(bec, efield=None, vel=None):
    """Eq. 29-30: (fext [3][N] or None, pdot [3] or None) from the BEC tensor [9][N]."""
    bec = _f64(bec)
    n = bec.shape[1]
    fext = np.zeros((3, n)) if efield is not None else None
    pdot = np.zeros(3) if vel is not None else None
    e = _f64(np.asarray(efield, dtype=np.float64)) if efield is not None else None
    v = _f64(vel) if vel is not None else None
    f = lib().orc_response
    f.restype = None
    f(C.c_int64(n), _p(bec), _p(e) if e is not None else None, _p(v) if v is not None else None,
      _p(fext) if fext is not None else None, _p(pdot) if pdot is not None else None)
    return fext, pdot


def compute_workload(w, **kw):
    if getattr(w, "zbl", None) is not None and "zbl" not in kw:
        kw["zbl"] = w.zbl
    return compute(w.model, w.params, w.es, w.pos, w.types, w.box, **kw)


def bspline5(dx):
    w = np.zeros(5)
    lib().orc_bspline5(C.c_double(dx), _p(w))
    return w


def alias_denominator(z):
    return float(lib().orc_alias_denominator(C.c_double(z)))


def fft3d(x, sign):
    """Unnormalised 3-D complex transform (sign -1 forward, +1 inverse)."""
    x = np.ascontiguousarray(x, dtype=np.complex128).copy()
    n0, n1, n2 = x.shape
    rc_ = lib().orc_fft3d(_p(x), C.c_int(n0), C.c_int(n1), C.c_int(n2), C.c_int(sign))
    assert rc_ == 0
    return x
