"""hydro_max_signal_speed_static: the max signal speed for callers that cannot allocate device memory.

Who that is: code that has no workspace to hand to hydro_bind_workspace and may not make one -- a hook that is given
somebody else's state inside their event loop, a process whose device memory all belongs to a framework's pool that
is full, a loop that must not call cudaMalloc because it synchronises the whole GPU.  The entry point reduces in a
512.25 KiB array built into the library (one per GPU, shared by every call, grids up to 65536 tiles of 64 x 4 x 1
cells), so what has to be shown is: (1) it gives what the workspace path (hydro_max_signal_speed) gives, (2) on two
calls in a row, the second on another state, so that nothing left in the shared array by the first call leaks into the
second, (3) it takes no device memory, and (4) it refuses grids beyond its limit with a text that says why.

This file is named test_zz_* so that pytest collects it LAST: `pytest -x` stops at the first failure, and a failure
here must not hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

from paper_1604_03360_b200 import workloads as W

pytestmark = pytest.mark.gpu

# the tolerance of test_max_signal_speed (test_gpu_parity.py): a few ulp
RTOL = 4e-15


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1604_03360_b200 import binding
    return binding


def workspace_path(B, w, precision):
    """The existing path: a bound context, hydro_set_state, hydro_max_signal_speed."""
    h = B.from_workload(w, precision=precision)
    v = h.max_signal_speed()
    h.close()
    return v


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("n", [(150, 21, 19), (64, 1, 1), (1, 33, 40), (48, 20, 1)])
def test_two_calls_in_a_row_match_the_workspace_path(B, n, precision):
    import torch
    shape = (n[2], n[1], n[0])
    # two different states: the first FASTER than the second, so a value surviving in the shared array would show
    fast = W.random_state(shape, seed=11, vmax=0.95)
    slow = W.random_state(shape, seed=12, vmax=0.3)
    want = []
    for cons in (fast, slow):
        w = W.Workload("rand", n, 0.1, (0, 0, 0), W.WENO5, (W.BC_OUTFLOW,) * 3, cons)
        want.append(workspace_path(B, w, precision))
    assert want[0] > want[1] > 0.0

    h = B.Hydro(n[0], n[1], n[2], 0.1, W.WENO5, precision=precision)      # never bound: there is no workspace
    dev = [torch.from_numpy(c).to(device="cuda", dtype=h.dtype).contiguous() for c in (fast, slow)]
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    h.max_signal_speed_static(dev[0], out[0:1])      # also the first call on this GPU in a fresh process (set-up)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    h.max_signal_speed_static(dev[0], out[0:1])
    h.max_signal_speed_static(dev[1], out[1:2])      # same stream: ordered after the first, as the header asks
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    got = out.cpu().numpy()
    for g, v in zip(got, want):
        assert abs(g - v) <= RTOL * v, (got, want)
    assert free1 >= free0, "the call took %d bytes of device memory" % (free0 - free1)
    # and once more on the first state: the array now holds the slow state's tiles
    h.max_signal_speed_static(dev[0], out[1:2])
    torch.cuda.synchronize()
    assert abs(float(out[1]) - want[0]) <= RTOL * want[0]
    h.close()


def test_largest_allowed_grid_and_the_first_one_beyond(B):
    """ceil(nx/64) * ceil(ny/4) * nz = 65536 tiles is served, one more z plane is refused before anything is launched."""
    import torch
    n = (4096, 4, 64)        # 64 * 1 * 64 = 4096 tiles ... a cheap shape; the limit itself follows
    n_max = (128, 8, 16384)  # 2 * 2 * 16384 = exactly 65536 tiles, 16.8 M cells
    for shape_n in (n, n_max):
        cons = W.random_state((shape_n[2], shape_n[1], shape_n[0]), seed=5, vmax=0.8)
        w = W.Workload("rand", shape_n, 0.1, (0, 0, 0), W.MUSTA_FORCE, (W.BC_OUTFLOW,) * 3, cons)
        want = workspace_path(B, w, 0)
        h = B.Hydro(shape_n[0], shape_n[1], shape_n[2], 0.1, W.MUSTA_FORCE)
        out = torch.zeros(1, dtype=torch.float64, device="cuda")
        h.max_signal_speed_static(torch.from_numpy(cons).cuda().contiguous(), out)
        assert abs(float(out[0]) - want) <= RTOL * want
        h.close()
    h = B.Hydro(128, 8, 16385, 0.1, W.MUSTA_FORCE)    # 65540 tiles
    small = torch.zeros(8, dtype=torch.float64, device="cuda")     # never read: the size check comes first
    rc = B.lib.hydro_max_signal_speed_static(h._h, small.data_ptr(), small.data_ptr())
    assert rc == B.EINVAL
    msg = B.lib.hydro_last_error(h._h).decode()
    assert "65540 tiles" in msg and "65536" in msg and "workspace" in msg, msg
    h.close()


def test_host_pointers_are_refused(B):
    import torch
    h = B.Hydro(16, 16, 16, 0.1, W.WENO5)
    host = np.zeros((5, 16, 16, 16))
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    rc = B.lib.hydro_max_signal_speed_static(h._h, ctypes.c_void_p(host.ctypes.data), out.data_ptr())
    assert rc == B.EINVAL and "device memory" in B.lib.hydro_last_error(h._h).decode()
    assert B.lib.hydro_max_signal_speed_static(h._h, None, out.data_ptr()) == B.EINVAL
    h.close()
