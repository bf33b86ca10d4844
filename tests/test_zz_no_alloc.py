"""qnep_neutralise_noalloc -- the entry point for callers that may not allocate device memory -- against the existing path.

Some users of this library cannot call cudaMalloc: a plug-in running inside an MD engine or an inference server whose own
pool has already taken the rest of the GPU (a raw allocation from a library would fail or eat memory the application
counted on), code in a section that must not stall the device (cudaMalloc / cudaFree may synchronise every stream), code
whose memory footprint is fixed before the first step.  For them include/qnep.h has one entry point, Eq. 33 of the paper
(charge neutralisation, PAPER.md :255-262), whose only scratch -- the partial sums of the raw charges -- is an array built
into the library.  All calls on a device share that array and it keeps the previous call's contents, so the test below
makes several calls in a row, of different sizes, and compares every one of them with what qnep_compute (which allocates
its workspace the usual way) returns for the same atoms, at the charge tolerance of the parity tests (1e-5 e).

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It passes alone in a fresh process and after the other tests (the one-off set-up happens in
whichever call comes first on the device)."""
import ctypes as C

import numpy as np
import pytest

import paper_2601_19034_b200 as Q
import qnep_inputs as I

TOL_Q = 1e-5          # e; the charge tolerance of tests/test_gpu_parity.py (BASELINE.json north_star)


@pytest.fixture(scope="module")
def lib():
    from paper_2601_19034_b200 import build
    build.build()
    return Q.load_library()


def existing_path(torch, w):
    """Charges after Eq. 33 and the raw network charges of the same atoms from qnep_compute (handle, allocated workspace)."""
    h = Q.from_workload(w)
    pos = torch.tensor(w.pos, dtype=torch.float64, device="cuda")
    types = torch.tensor(w.types, dtype=torch.int32, device="cuda")
    try:
        out = h.compute(pos, types, w.box, want=Q.WANT_CHARGES)
    except Q.QnepError as err:          # documented protocol: the handle has grown its lists, call again
        if err.code != Q.QNEP_ERR_NEIGHBOR_OVERFLOW:
            raise
        out = h.compute(pos, types, w.box, want=Q.WANT_CHARGES)
    q_raw = h.debug_copy(Q.DBG_Q_RAW, (w.n_atoms,))
    charges = out["charges"].clone()
    h.destroy()
    return q_raw, charges


@pytest.mark.gpu
def test_noalloc_matches_existing_path_on_calls_in_a_row(lib):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    # 26 112 atoms (26 partial sums), then 512 atoms (one: slots 1..25 still hold the first call's sums), then the large one again
    cases = [I.config2(), I.config0(), I.config2()]
    refs = [existing_path(torch, w) for w in cases[:2]]
    refs.append(refs[0])
    torch.cuda.synchronize()
    outs = []
    for k, (w, (q_raw, _)) in enumerate(zip(cases, refs)):     # back to back on one stream, nothing in between
        if k < 2:
            outs.append(Q.neutralise_noalloc(q_raw, w.model.q_total, out=torch.full_like(q_raw, float("nan"))))
        else:                                                  # in place: the output buffer is the input buffer
            buf = q_raw.clone()
            assert Q.neutralise_noalloc(buf, w.model.q_total, out=buf) is buf
            outs.append(buf)
    torch.cuda.synchronize()
    for k, (w, (q_raw, charges), got) in enumerate(zip(cases, refs, outs)):
        d = float((got - charges).abs().max())
        total = float(got.sum())
        print(f"[noalloc call {k}: {w.name}] N={w.n_atoms} max |dq| vs qnep_compute = {d:.2e} e, sum q = {total:.2e}")
        assert torch.isfinite(got).all()
        assert d <= TOL_Q, d
        assert abs(total - w.model.q_total) <= 1e-9 * w.n_atoms      # Eq. 33: the charges add up to Q
        # every atom received the same shift
        shift = (got - q_raw).cpu().numpy()
        assert np.ptp(shift) <= 1e-14, np.ptp(shift)            # up to the rounding of q_raw + shift
    assert torch.equal(outs[0], outs[2])                        # the same input gives the same bits, whatever ran in between


@pytest.mark.gpu
def test_noalloc_at_its_maximum_size_and_ragged_tails(lib):
    """Exactly QNEP_NOALLOC_MAX_ATOMS atoms (all 4096 partial sums in use), then sizes around the 1024-atom block and the
    256-thread edges, against the definition of Eq. 33 evaluated with torch in fp64 on the same device."""
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    gen = torch.Generator(device="cuda").manual_seed(20260119034)
    for n in (Q.NOALLOC_MAX_ATOMS, 1, 255, 256, 257, 1023, 1024, 1025, 4097, Q.NOALLOC_MAX_ATOMS - 1):
        q_raw = torch.randn(n, dtype=torch.float64, device="cuda", generator=gen) * 0.4
        q_total = -1.0 if n % 2 else 2.0
        got = Q.neutralise_noalloc(q_raw, q_total)
        want = q_raw + (q_total - q_raw.sum()) / n
        d = float((got - want).abs().max())
        assert d <= 1e-12, (n, d)                                   # both in fp64; only the order of the sum differs
        assert abs(float(got.sum()) - q_total) <= 1e-9
    with pytest.raises(Q.QnepError) as ei:                          # one atom more than the built-in array serves
        Q.neutralise_noalloc(torch.zeros(Q.NOALLOC_MAX_ATOMS + 1, dtype=torch.float64, device="cuda"), 0.0)
    assert ei.value.code == Q.QNEP_ERR_UNSUPPORTED and "QNEP_NOALLOC_MAX_ATOMS" in str(ei.value)


def test_noalloc_rejects_bad_sizes_before_touching_the_gpu(lib):
    # the argument checks come before any CUDA call, so this runs without a device; the pointers are never dereferenced
    msg = C.create_string_buffer(512)
    dummy = C.c_void_p(256)
    rc = lib.qnep_neutralise_noalloc(Q.NOALLOC_MAX_ATOMS + 1, dummy, 0.0, dummy, None, msg, len(msg))
    assert rc == Q.QNEP_ERR_UNSUPPORTED
    text = msg.value.decode()
    assert str(Q.NOALLOC_MAX_ATOMS + 1) in text and "QNEP_NOALLOC_MAX_ATOMS" in text and str(Q.NOALLOC_MAX_ATOMS) in text
    assert lib.qnep_neutralise_noalloc(0, dummy, 0.0, dummy, None, msg, len(msg)) == Q.QNEP_ERR_INVALID_ARG
    assert b"n_atoms" in msg.value
    assert lib.qnep_neutralise_noalloc(10, None, 0.0, dummy, None, msg, len(msg)) == Q.QNEP_ERR_INVALID_ARG
    assert lib.qnep_neutralise_noalloc(10, dummy, 0.0, None, None, None, 0) == Q.QNEP_ERR_INVALID_ARG     # no message buffer is fine
    header = open(Q.LIB_PATH.replace("paper_2601_19034_b200/libqnep_b200.so", "include/qnep.h")).read()
    assert f"#define QNEP_NOALLOC_MAX_ATOMS {Q.NOALLOC_MAX_ATOMS}" in header
