"""corr_accumulate_wide_static -- the entry point for callers that may not allocate device memory.

Some users of this library cannot call cudaMalloc while they run: a correlator's real-time loop cannot take the
device-wide stall of cudaMalloc / cudaFree inside its sample-rate deadline, and a plug-in inside a host application that
has given the whole GPU to its own memory pool has nothing left to allocate from (or is forbidden to after start-up).
For them the library carries a fixed 16 MiB device array (CORR_STATIC_BATCH_BYTES) that stands in for the batch buffer
corr_accumulate_wide allocates on first use.  The array is shared by every call on a GPU and keeps the last call's
contents, so these tests run two calls in a row (the second finds the first one's batch in the buffer, and a smaller
third shape finds a larger shape's leftovers) and compare against the allocating path, which the accumulate tests pin
to the oracle: the integer results must be identical bit for bit; the float path adds its time slices with atomic
adds in whatever order they finish, so two runs of the SAME entry point already differ in the last bits, and the float
case is held to the parity tests' own tolerance, |delta| <= 1e-5 sqrt(|V_ii V_jj|) (tests/parity_util.py).

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It must pass alone in a fresh process (first call = address look-up) and after all other tests."""
from __future__ import annotations

import numpy as np
import pytest

import corrgen
from parity_util import f32_tolerance_check

pytestmark = pytest.mark.gpu


def _input(dtype, N, C, T, seed):
    import torch
    if dtype == "cf32":
        x = np.random.default_rng(seed).standard_normal((T, C, N, 2)).astype(np.float32)
        return torch.from_numpy(x).cuda()
    rng = np.random.default_rng(seed)
    x = rng.integers(-127, 128, size=(T, C, N, 2), dtype=np.int8)
    if dtype == "ci4":
        x = corrgen.pack_ci4(np.clip(x, -8, 7).astype(np.int8))
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


# (dtype, N_I, C, T): a multi-tile int8 shape with a ragged K tail, a 2-channels-per-tile shape, a time-sliced plan
# (few channels, long T: the path that clears its output before filling it), the 4-bit mode and the float path
SHAPES = [("ci8", 128, 5, 333), ("ci8", 32, 6, 97), ("ci8", 64, 3, 20000), ("ci4", 64, 4, 130), ("cf32", 64, 5, 61)]


@pytest.mark.parametrize("dtype,N,C,T", SHAPES)
def test_static_buffer_path_equals_allocating_path_on_two_calls_in_a_row(dtype, N, C, T):
    import torch
    import paper_0906_1887_b200 as corr
    h = corr.corr_create(N, C, T, dtype)
    try:
        assert h.vis_bytes <= corr.CORR_STATIC_BATCH_BYTES
        batches = [_input(dtype, N, C, T, seed) for seed in (11, 12)]
        acc_ref, acc_new = h.empty_acc(), h.empty_acc()
        for k, x in enumerate(batches):          # two calls in a row on the shared buffer, no host sync between them
            h.accumulate_wide_static(x, acc_new)
            h.accumulate_wide(x, acc_ref)
            torch.cuda.synchronize()
            if dtype == "cf32":
                f32_tolerance_check(acc_new.cpu().numpy(), acc_ref.cpu().numpy(), N, rel=1e-5)
            else:
                assert torch.equal(acc_new, acc_ref), f"after call {k + 1}"
        assert acc_ref.abs().sum().item() > 0    # the comparison is not of two untouched buffers
        if dtype != "cf32":                      # the read-out of either accumulator is the same too
            assert torch.equal(h.normalize_wide(acc_new, 2 * T), h.normalize_wide(acc_ref, 2 * T))
    finally:
        corr.corr_destroy(h)


def test_static_buffer_path_on_a_side_stream_and_with_accumulate_mode_left_alone():
    """The call is asynchronous on the caller's stream and does not disturb corr_set_accumulate's state."""
    import torch
    import paper_0906_1887_b200 as corr
    N, C, T = 96, 4, 257
    h = corr.corr_create(N, C, T, "ci8")
    try:
        x0, x1 = _input("ci8", N, C, T, 21), _input("ci8", N, C, T, 22)
        want = h.empty_acc()
        h.accumulate_wide(x0, want)
        h.accumulate_wide(x1, want)
        torch.cuda.synchronize()
        h.set_accumulate(True)
        s = torch.cuda.Stream()
        acc = h.empty_acc()
        torch.cuda.synchronize()
        with torch.cuda.stream(s):
            h.accumulate_wide_static(x0, acc, stream=s)
            h.accumulate_wide_static(x1, acc, stream=s)
        s.synchronize()
        assert torch.equal(acc, want)
        assert h.accumulate_count == 0         # the batches were overwriting integrations, not accumulate-mode ones
    finally:
        corr.corr_destroy(h)


def test_static_buffer_path_rejects_a_batch_larger_than_the_buffer():
    import torch
    import paper_0906_1887_b200 as corr
    N, C, T = 256, 64, 32                        # 64 * 32896 * 8 B = 16.06 MiB > 16 MiB
    h = corr.corr_create(N, C, T, "ci8")
    try:
        assert h.vis_bytes > corr.CORR_STATIC_BATCH_BYTES
        x = torch.zeros((T, C, N, 2), dtype=torch.int8, device="cuda")
        acc = h.empty_acc()
        with pytest.raises(corr.CorrError) as e:
            h.accumulate_wide_static(x, acc)
        assert e.value.status == corr.CORR_EUNSUPPORTED and "CORR_STATIC_BATCH_BYTES" in str(e.value)
        torch.cuda.synchronize()
        assert acc.abs().sum().item() == 0       # nothing was enqueued
        h.accumulate_wide(x, acc)                # the allocating path still serves the shape
        torch.cuda.synchronize()
    finally:
        corr.corr_destroy(h)
