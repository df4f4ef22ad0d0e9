"""shasta_conserved_totals_static (include/shasta.h): the conserved totals of eqs. (12)-(14), through the
entry point that allocates nothing (its block partial sums live in a file-scope device array), against the handle's
shasta_conserved_totals on the same fields.  Collected last on purpose (the run uses -x); passes alone in a
fresh process and after the other GPU tests.  Tolerance: that of test_conserved_totals_periodic, 1e-12 of the energy."""
import ctypes as C

import numpy as np
import pytest

from paper_1206_0919_b200 import inputs

pytestmark = pytest.mark.gpu

REL = 1e-12


@pytest.fixture(scope="module", autouse=True)
def _built():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1206_0919_b200 import build
    build.build()


def _handle_totals(c):
    """existing path: the state goes into a handle; its totals and its conserved fields (device tensors)"""
    import torch
    from paper_1206_0919_b200.shasta import Shasta
    s = Shasta(c["nx"], c["ny"], c["nz"], c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"])
    s.set_state(*[torch.from_numpy(c[k]).cuda() for k in ("e", "n", "vx", "vy", "vz")])
    U = s.get_conserved()
    t = np.array(s.conserved_totals())
    s.close()
    return t, [U[k] for k in ("E", "Mx", "My", "Mz", "R")]


def _close(got, ref):
    return np.max(np.abs(got - ref)) <= REL * abs(ref[0])


def test_static_totals_match_the_handle_path_on_calls_in_a_row():
    import torch
    from paper_1206_0919_b200 import shasta as sh
    # A: 16 169 cells, one ragged block.  B: 336 000 cells, 21 blocks, ragged tail.  Then A again: the array still
    # holds B's 21 partial sums and only the first may be read.
    cA = inputs.random_state(37, 19, 23, seed=5, kind="rough")
    cB = inputs.random_state(96, 70, 50, seed=6, kind="smooth")
    refA, UA = _handle_totals(cA)
    refB, UB = _handle_totals(cB)
    out = torch.full((3, 5), float("nan"), dtype=torch.float64, device="cuda")
    sh.conserved_totals_static(*UA, cA["dx"] ** 3, out[0])          # set-up call: symbol address of this device
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    out.fill_(float("nan"))
    sh.conserved_totals_static(*UA, cA["dx"] ** 3, out[0])
    sh.conserved_totals_static(*UB, cB["dx"] ** 3, out[1])
    sh.conserved_totals_static(*UA, cA["dx"] ** 3, out[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0, "device memory was allocated by the static entry point"
    got = out.cpu().numpy()
    assert _close(got[0], refA), (got[0], refA)
    assert _close(got[1], refB), (got[1], refB)
    assert _close(got[2], refA), (got[2], refA)
    assert np.array_equal(got[0], got[2])                            # same grid, same order: same bits
    # and against a plain sum of the same fields (fp64, other order)
    plain = np.array([float(u.sum()) for u in UB]) * cB["dx"] ** 3
    assert np.max(np.abs(got[1] - plain)) <= 1e-11 * abs(plain[0])


def test_static_totals_on_a_side_stream_and_many_blocks():
    import torch
    from paper_1206_0919_b200 import shasta as sh
    c = inputs.hotspots(128, steps=0)
    ref, U = _handle_totals(c)                                       # 2^21 cells: 128 blocks
    out = torch.empty(5, dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        sh.conserved_totals_static(*U, c["dx"] ** 3, out, stream=st)
    st.synchronize()
    assert _close(out.cpu().numpy(), ref)


def test_static_totals_limits():
    import torch
    from paper_1206_0919_b200 import shasta as sh
    L = sh.load()
    nmax = sh.conserved_totals_static_max_cells()
    assert nmax == 1 << 26
    u = torch.ones(8, dtype=torch.float64, device="cuda")
    out = torch.full((5,), 7.0, dtype=torch.float64, device="cuda")
    p = C.c_void_p(u.data_ptr())
    # beyond the static array: refused before anything is launched or read
    rc = L.shasta_conserved_totals_static(nmax + 1, p, p, p, p, p, 1.0, C.c_void_p(out.data_ptr()), None)
    assert rc == -1 and b"exceeds" in L.shasta_last_error(None)
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [7.0] * 5
    rc = L.shasta_conserved_totals_static(8, p, p, None, p, p, 1.0, C.c_void_p(out.data_ptr()), None)
    assert rc == -1 and b"NULL" in L.shasta_last_error(None)
    rc = L.shasta_conserved_totals_static(8, p, p, p, p, p, 1.0, None, None)
    assert rc == -1
    # no cells: zeros;  8 cells of 1 with dv = 0.5: 4
    sh.conserved_totals_static(u[:0], u[:0], u[:0], u[:0], u[:0], 1.0, out)
    assert out.cpu().tolist() == [0.0] * 5
    sh.conserved_totals_static(u, u, u, u, u, 0.5, out)
    assert out.cpu().tolist() == [4.0] * 5
