"""tdse_dissimilarity_static: eq (16) through the entry point that allocates nothing.

Why the library has it: tdse_dissimilarity() takes its reduction buffer from cudaMalloc.  A caller that has given
almost all of HBM to the grids (the fill-HBM configuration), a process whose device memory is owned by a single pool
with a hard cap, or a loop that cannot take the device-wide stall of cudaMalloc / cudaFree while other streams are
stepping, cannot use that.  The static variant keeps the same two kernels and puts the partial sums in a fixed 2 MiB
array inside libtdse.so; inputs and outputs are the caller's own device buffers.

What is checked: the result equals the allocating path's (same tolerance as the reduction check in
test_gpu_parity.py, 1e-12 relative) on calls made back to back -- with a different batch and window in between, so the
second call finds the first call's leftovers laid out differently in the shared array, and then the first call again;
sizes over the limit are refused with a message; device memory in use does not grow across the calls.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It does not depend on anything they leave behind (fresh context, own tensors) and passes alone as well.
"""
import numpy as np
import pytest

from workloads import make_config

pytestmark = pytest.mark.gpu

RTOL = 1e-12      # test_gpu_parity.py: "the reduction alone ... rounding level"


def close(got, want):
    return np.all(np.abs(got - want) <= RTOL * np.abs(want))


def test_static_scratch_dissimilarity_matches_the_allocating_path_on_repeated_calls():
    import torch
    from paper_2401_07416_b200 import (Tdse, TdseError, TDSE_EINVAL, TDSE_STATIC_SCRATCH_DOUBLES,
                                       dissimilarity_static)
    w = make_config(3, n=(40, 36, 44), batch=10, steps=40, dtype="f32").with_(every=5)
    t = Tdse.from_workload(w)
    nfr = w.steps // w.every + 1
    t.set_frames(nfr, True)
    t.step(w.steps)
    assert t.get_info("nframes") == nfr
    dA = w.dx ** 2

    # the existing path, on two windows
    s0, s1 = 1, nfr - 2
    want_a = t.dissimilarity(s0, s1)
    want_b = t.dissimilarity(0, nfr - 1)
    assert np.all(want_a[np.triu_indices(w.batch, 1)] > 0.0)

    # caller-owned input and outputs (the frames come back through the ABI and go up again as a plain tensor)
    host = np.stack([t.frames_read(b) for b in range(w.batch)])            # [batch][nfr][ny][nx]
    frames = torch.from_numpy(host).to("cuda:0")
    sub = frames[:7].contiguous()                                          # another batch: other offsets in the scratch
    out_a = torch.full((w.batch, w.batch), -1.0, dtype=torch.float64, device="cuda:0")
    out_b = torch.full((7, 7), -1.0, dtype=torch.float64, device="cuda:0")
    out_c = torch.full((w.batch, w.batch), -1.0, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()

    dissimilarity_static(frames, s0, s1, dA, out_a)                        # first call on this GPU: address look-up
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    dissimilarity_static(sub, 0, nfr - 1, dA, out_b)                       # second call, straight after, other shape
    dissimilarity_static(frames, s0, s1, dA, out_c)                        # and the first one again
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before                                       # nothing was allocated on the device

    got_a, got_b, got_c = out_a.cpu().numpy(), out_b.cpu().numpy(), out_c.cpu().numpy()
    assert close(got_a, want_a) and np.array_equal(got_a, got_a.T) and np.all(np.diag(got_a) == 0.0)
    assert close(got_b, want_b[:7, :7]) and np.array_equal(got_b, got_b.T) and np.all(np.diag(got_b) == 0.0)
    assert np.array_equal(got_c, got_a)                                    # the call in between left no trace

    # beyond the fixed array: refused with a message, output untouched
    big = int(np.sqrt(TDSE_STATIC_SCRATCH_DOUBLES)) + 1                    # big*big*1 frames > limit
    tiny = torch.zeros((big, 1, 2, 2), dtype=torch.float64, device="cuda:0")
    out_big = torch.full((big, big), -1.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(TdseError) as e:
        dissimilarity_static(tiny, 0, 0, dA, out_big)
    assert e.value.code == TDSE_EINVAL and "exceeds the fixed scratch" in str(e.value)
    assert torch.all(out_big == -1.0)
    # exactly at the limit is accepted: 512 * 512 * 1 = 262144
    edge = big - 1
    assert edge * edge == TDSE_STATIC_SCRATCH_DOUBLES
    dissimilarity_static(tiny[:edge].contiguous(), 0, 0, dA, out_big[:edge, :edge].contiguous())
    torch.cuda.synchronize()
    # a host pointer is refused instead of faulting in the kernel
    with pytest.raises(TdseError) as e:
        dissimilarity_static(torch.zeros((2, 1, 2, 2), dtype=torch.float64), 0, 0, dA, out_big)
    assert e.value.code == TDSE_EINVAL
    t.close()
