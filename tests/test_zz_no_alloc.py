"""xy_measure_static: the observable reduction for callers that cannot allocate device memory.

Some users of this library hold a spin state on the GPU but have no way to obtain more device memory when they
want its observables: a monitoring hook that a running simulation lends its state buffer to after the simulation
handed the rest of the card to its own pool; a loop that may not stall and therefore may not call cudaMalloc /
cudaFree (both synchronise the device); a process with a memory budget fixed at start-up.  Every other path of
the library needs an xy_ctx with a workspace that somebody must allocate.  For those users the library carries
1 MiB of scratch compiled into it and xy_measure_static, which uses it and allocates nothing.

What is checked here, against the existing path (xy_measure on a context, rows mapped from rank to slot) and at
the tolerance all observable tests use (P3: |dE| <= 1e-6 * 3N, |dMx|, |dMy| <= 1e-6 * N; tests/parity.py):
  * two calls in a row on the same system, the state and the labels changed in between;
  * calls of different shapes back to back, so that the second finds the first's leftovers in the shared
    scratch (nothing is cleared between calls: every entry read is written first);
  * no device memory disappears during a call once the device has been set up;
  * shapes that need more than the built-in 1 MiB, and malformed arguments, are refused before anything is
    touched (these run without a GPU).

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
It passes alone in a fresh process (the first call then does the per-device set-up) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1211_0780_b200 import inputs
from . import parity as P

SEED = inputs.SEED
SCRATCH_BYTES = 1 << 20           # XY_STATIC_SCRATCH_BYTES of include/xy.h


def by_slot(obs_rank, slot_at_rank):
    """xy_measure reports by rank, xy_measure_static by slot: obs_slot[slot_at_rank[k]] = obs_rank[k]."""
    out = np.empty_like(obs_rank)
    out[np.asarray(slot_at_rank)] = obs_rank
    return out


def static_obs(xy, out):
    import torch
    got = xy.measure_static(out)
    assert got is out
    torch.cuda.synchronize()
    return out.cpu().numpy()


# several tiles in y and z, ragged rows (L/8 = 1, 3, 5, 10 float4), one replica, the headline lattice size
@pytest.mark.gpu
@pytest.mark.parametrize("L,R", [(8, 8), (24, 5), (32, 16), (40, 1), (64, 4), (80, 3), (160, 2)])
def test_static_reduction_equals_measure_on_two_calls_in_a_row(xy_mod, L, R):
    import torch
    N = L ** 3
    xy = xy_mod.XY(L, R, inputs.beta_ladder(0.44, 0.47, R), SEED)
    out = torch.full((R, 5), float("nan"), dtype=torch.float64, device="cuda")
    # call 1: a partially ordered state (M of order N, so Mx, My, |M|^2 are all exercised)
    xy.set_state(inputs.smooth_state(L, R, 21))
    want = by_slot(xy.measure(), xy.get_perm())
    got = static_obs(xy, out)
    print(L, R, "call 1", P.check_observables(got, want, N))
    # call 2, straight after: new spins and, where R > 1, new labels (the static call ignores them by design)
    xy.metropolis_sweep()
    xy.pt_exchange(); xy.pt_exchange()
    if R >= 3:
        xy.set_perm(np.roll(xy.get_perm(), 1))
    free_before = torch.cuda.mem_get_info()[0]
    got2 = static_obs(xy, out)
    assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was allocated during xy_measure_static"
    want2 = by_slot(xy.measure(), xy.get_perm())
    print(L, R, "call 2", P.check_observables(got2, want2, N))
    assert not np.array_equal(got, got2)                 # the second call really reduced the new state
    # the reduction is deterministic: a third call returns the second's bits
    assert np.array_equal(static_obs(xy, out), got2)
    xy.close()


@pytest.mark.gpu
def test_static_reduction_ignores_what_the_previous_call_left_in_the_scratch(xy_mod):
    """Big shape, small shape, big shape, on one stream: each call overwrites exactly the entries it reads."""
    import torch
    big = xy_mod.XY(64, 6, inputs.beta_ladder(0.44, 0.47, 6), SEED)
    small = xy_mod.XY(16, 2, inputs.beta_ladder(0.44, 0.47, 2), SEED + 1)
    big.set_state(inputs.uniform_state(64, 6, 31)); small.set_state(inputs.smooth_state(16, 2, 32))
    ob = torch.empty((6, 5), dtype=torch.float64, device="cuda")
    os_ = torch.empty((2, 5), dtype=torch.float64, device="cuda")
    for xy, out in ((big, ob), (small, os_), (big, ob), (small, os_)):
        got = static_obs(xy, out)
        P.check_observables(got, by_slot(xy.measure(), xy.get_perm()), xy.N)
    # a closed form, so that the check does not rest on the other CUDA path alone: all spins at one angle
    small.init_ordered(1.25)
    got = static_obs(small, os_)
    n = float(small.N)
    assert np.allclose(got[:, 0], -3.0 * n, rtol=0, atol=1e-6 * 3 * n)
    assert np.allclose(got[:, 1], n * np.cos(1.25), rtol=0, atol=1e-6 * n)
    assert np.allclose(got[:, 2], n * np.sin(1.25), rtol=0, atol=1e-6 * n)
    big.close(); small.close()


@pytest.mark.gpu
def test_static_reduction_refuses_pointers_it_cannot_use(xy_mod):
    import torch
    lib = xy_mod.load_library()
    st = torch.zeros(8 * 512, dtype=torch.float32, device="cuda")
    out = torch.zeros(8 * 5, dtype=torch.float64, device="cuda")
    host = np.zeros(8 * 512, dtype=np.float32)
    s = torch.cuda.current_stream().cuda_stream
    assert lib.xy_measure_static(st.data_ptr(), 8, 8, out.data_ptr(), s) == 0
    assert lib.xy_measure_static(host.ctypes.data & ~15, 8, 8, out.data_ptr(), s) == -1        # pageable host memory
    assert lib.xy_measure_static(st.data_ptr() + 4, 8, 8, out.data_ptr(), s) == -1             # misaligned
    assert lib.xy_measure_static(st.data_ptr(), 8, 8, None, s) == -1
    torch.cuda.synchronize()
    assert np.allclose(out.cpu().numpy().reshape(8, 5), [[-3.0 * 512, 512.0, 0.0, 512.0 ** 2, 512.0 ** 4]] * 8)


def test_static_reduction_refuses_sizes_beyond_its_scratch(xy_mod):
    """No GPU needed: the shape and size checks come before the library touches the device (the pointers are
    never dereferenced).  24 bytes per replica and tile: L = 8 has one tile, so R = 43690 is the last that fits."""
    lib = xy_mod.load_library()
    dummy = C.c_void_p(0x1000)
    assert 24 * 43690 <= SCRATCH_BYTES < 24 * 43691
    rc = lib.xy_measure_static(dummy, 8, 43691, dummy, None)
    msg = lib.xy_last_error().decode()
    assert rc == -1 and "scratch" in msg and str(24 * 43691) in msg and str(SCRATCH_BYTES) in msg, msg
    assert lib.xy_measure_static(dummy, 8, 65535, dummy, None) == -1
    for L, R in ((7, 8), (12, 8), (0, 1), (8, 0), (2048, 1), (8, 65536)):
        assert lib.xy_measure_static(dummy, L, R, dummy, None) == -1, (L, R)
        assert b"xy_measure_static" in lib.xy_last_error()
    assert lib.xy_measure_static(None, 8, 8, dummy, None) == -1 and b"NULL" in lib.xy_last_error()
