"""sim_cfl_dt_static: the CFL time step for callers that must not allocate device memory.

Some users of this library cannot call cudaMalloc when they need a time step: the host framework's
pool allocator owns the GPU's memory, or they sit in a loop where cudaMalloc's device-wide
synchronisation is not acceptable, or they are a plug-in that only receives pointers to the host
solver's fields.  For them the library has one entry point whose scratch memory is a fixed array
inside the library itself (include/floodped.h).  This file checks it against the path everybody
else uses -- the time step a handle derives on the device (flood kernel's fused reduction ->
tail kernel, read with sim_get_stats) -- on the same flood state, twice in a row, because the
array is shared by all calls and keeps what the call before left in it.

The file is named so that pytest collects it last: with `-x` a failure here hides nothing.  It
passes alone in a fresh process (the first call on the device does the one-time address look-up)
and after the rest of the suite (the look-up then happens with many handles created and gone).
"""
import ctypes as C

import numpy as np
import pytest

from paper_1908_05232_b200 import binding, scenarios as S

# dt of the next step is compared at 10 * TOL everywhere in the GPU suite (tests/test_gpu_parity.py)
TOL = {64: 1e-12, 32: 1e-5}


def _device_state(g, sc, torch):
    """(h, qx, qy, mask) of the handle's current level as torch CUDA tensors: what a caller that
    holds its fields on the device would pass."""
    tdt = torch.float64 if sc.real_bits == 64 else torch.float32
    h, qx, qy = (torch.empty(sc.nx * sc.ny, dtype=tdt, device="cuda") for _ in range(3))
    g.read_conserved_into(h.data_ptr(), qx.data_ptr(), qy.data_ptr())
    mask = None if sc.mask is None else torch.from_numpy(np.ascontiguousarray(sc.mask, np.uint8)).cuda()
    return h, qx, qy, mask


def _static_dt(sc, h, qx, qy, mask, out, torch):
    binding.cfl_dt_static(h.data_ptr(), qx.data_ptr(), qy.data_ptr(), None if mask is None else mask.data_ptr(),
                          h.numel(), sc.real_bits, sc.dx, sc.dy, sc.g, sc.h_dry, sc.cfl,
                          sc.dt_max, torch.cuda.current_stream().cuda_stream, out.data_ptr())


@pytest.mark.gpu
@pytest.mark.parametrize("bits", [32, 64])
def test_static_scratch_time_step_matches_the_handle_twice_in_a_row(bits):
    import torch

    # Config 2's hall (solid shops, dry start, breach inflow) on a 200 x 200 grid: four full 8192-cell blocks and a
    # ragged fifth; flood agents only (the time step is theirs), inflow strong enough that the CFL bound is active
    sc = S.make(2, n=200, q_peak=40.0)
    sc.real_bits = bits                   # the binding converts the arrays to the precision named here
    sc.dt_max = 1.0                       # stated, so that both sides clamp to the same number
    assert sc.nx * sc.ny > 3 * 8192 and (sc.nx * sc.ny) % 8192 != 0
    g = binding.Sim(sc, with_peds=False)
    out = torch.full((2, 2), -1.0, dtype=torch.float64, device="cuda")
    seen = []
    for call, steps in enumerate((60, 40)):
        g.step(steps)
        want = g.stats()["dt"]            # synchronises; the handle's own time step for the next step
        h, qx, qy, mask = _device_state(g, sc, torch)
        _static_dt(sc, h, qx, qy, mask, out[call], torch)
        torch.cuda.synchronize()
        lam, dt = out[call].tolist()
        assert lam > 0.0 and 0.0 < dt < sc.dt_max, (lam, dt)          # water is moving: the CFL bound is the active one
        assert abs(dt - want) <= 10 * TOL[bits] * want, (call, dt, want)
        assert abs(dt - sc.cfl / lam) <= 1e-15 * dt
        seen.append(dt)
    assert seen[0] != seen[1]              # two different states: the second answer is not the first one's leftovers
    # same inputs again, back to back on one stream with no synchronisation between the calls
    again = torch.full((2, 2), -1.0, dtype=torch.float64, device="cuda")
    _static_dt(sc, h, qx, qy, mask, again[0], torch)
    _static_dt(sc, h, qx, qy, mask, again[1], torch)
    torch.cuda.synchronize()
    assert again[0].tolist() == out[1].tolist() and again[1].tolist() == out[1].tolist()
    g.close()


@pytest.mark.gpu
def test_static_scratch_dry_state_and_empty_input_give_dt_max():
    import torch

    h = torch.zeros(20000, dtype=torch.float32, device="cuda")
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    for n in (20000, 0):
        out.fill_(-1.0)
        binding.cfl_dt_static(h.data_ptr(), h.data_ptr(), h.data_ptr(), None, n, 32, 1.0, 1.0, 9.81, 1e-3, 0.5, 0.125,
                              None, out.data_ptr())
        torch.cuda.synchronize()
        assert out.tolist() == [0.0, 0.125]
    # one wet cell at rest, in the ragged tail of the last block: lam = sqrt(g h) / dx exactly as fp32 computes it
    h[19999] = 2.0
    binding.cfl_dt_static(h.data_ptr(), torch.zeros_like(h).data_ptr(), torch.zeros_like(h).data_ptr(), None, 20000, 32,
                          0.5, 1.0, 9.81, 1e-3, 0.5, 10.0, None, out.data_ptr())
    torch.cuda.synchronize()
    lam = float(np.sqrt(np.float32(9.81) * np.float32(2.0), dtype=np.float32) * np.float32(2.0))
    assert out.tolist() == [lam, 0.5 / lam]
    # a solid mask takes the cell out again
    mask = torch.zeros(20000, dtype=torch.uint8, device="cuda"); mask[19999] = 1
    z = torch.zeros_like(h)
    binding.cfl_dt_static(h.data_ptr(), z.data_ptr(), z.data_ptr(), mask.data_ptr(), 20000, 32, 0.5, 1.0, 9.81, 1e-3, 0.5,
                          10.0, None, out.data_ptr())
    torch.cuda.synchronize()
    assert out.tolist() == [0.0, 10.0]


def test_static_scratch_refuses_sizes_beyond_its_array():
    """No GPU needed: the size check comes before any CUDA call, and names the limit."""
    from paper_1908_05232_b200 import build
    build.build()
    L = binding.load_library()
    dummy = C.c_void_p(256)
    rc = L.sim_cfl_dt_static(dummy, dummy, dummy, None, binding.SIM_CFL_STATIC_MAX_CELLS + 1, 32, 1.0, 1.0, 9.81, 1e-3, 0.5,
                             1.0, None, dummy)
    assert rc == binding.SIM_EINVAL
    msg = L.sim_last_error(None).decode()
    assert "SIM_CFL_STATIC_MAX_CELLS" in msg and str(1 << 28) in msg
    assert L.sim_cfl_dt_static(dummy, dummy, dummy, None, 10, 16, 1.0, 1.0, 9.81, 1e-3, 0.5, 1.0, None, dummy) == binding.SIM_EINVAL
    assert L.sim_cfl_dt_static(dummy, dummy, dummy, None, 10, 32, 1.0, 1.0, 9.81, 1e-3, 0.5, 1.0, None, None) == binding.SIM_EINVAL
    with pytest.raises(binding.FloodpedError):
        binding.cfl_dt_static(256, 256, 256, None, -1, 32, 1.0, 1.0, 9.81, 1e-3, 0.5, 1.0, None, 256)
