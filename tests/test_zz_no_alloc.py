"""uep_histogram_static: the histogram entry point that allocates nothing (its scratch is a fixed
array in the library's device image, include/uep.h).  Collected last on purpose (file name): the
suite runs with `pytest -x`, a failure here must not hide another test.

The GPU test compares it, bit for bit (integer work: the tolerance of every parity test here is
zero), with the existing path — uep_histogram through a context and a workspace — on two calls in
a row that share the static array: a large input, then a smaller ragged one with another expert
count and ids outside [0, E), so that rows or columns left over from the first call would show.
It runs the same alone in a fresh process and behind the other tests: it depends on no state but
the array, which every call rewrites before reading."""
import ctypes

import numpy as np
import pytest
import torch

import oracle
from paper_2606_04101_b200 import binding, synth


def _existing_path(ids, E, R):
    T, k = ids.shape
    ctx = binding.Context(T, k, E, R, 1, 64, gate_dtype=binding.GATE_NONE)
    ws = ctx.new_workspace()
    count = torch.full((E,), -7, dtype=torch.int32, device="cuda")
    ctx.uep_histogram(ids, count, ws)
    torch.cuda.synchronize()
    out = count.cpu().numpy()
    ctx.close()
    return out


@pytest.mark.gpu
def test_static_histogram_matches_the_existing_path_twice_in_a_row():
    binding.uep_histogram_static_setup()
    # call 1: the benchmarked shape (2 Mi slots, E = 256); call 2: 3 x 33 331 = 99 993 slots
    # (ragged: not a multiple of 4, fewer CTAs than call 1), E = 160, some ids invalid
    ids1 = synth.zipf_topk_ids(262144, 8, 256, 1.0, 4101, device="cuda")
    ids2 = synth.zipf_topk_ids(33331, 3, 160, 1.4, 4102, device="cuda")
    bad = torch.arange(0, ids2.numel(), 977, device="cuda")
    ids2.view(-1)[bad] = torch.where(bad % 2 == 0, torch.tensor(-1, device="cuda"), torch.tensor(160, device="cuda")).to(torch.int32)
    want1, want2 = _existing_path(ids1, 256, 64), _existing_path(ids2, 160, 32)
    out1 = torch.full((256,), -7, dtype=torch.int32, device="cuda")
    out2 = torch.full((160,), -7, dtype=torch.int32, device="cuda")
    out3 = torch.full((256,), -7, dtype=torch.int32, device="cuda")
    empty = torch.full((16,), -7, dtype=torch.int32, device="cuda")
    binding.uep_histogram_static(ids1, 256, out3)          # warm: module load, address resolved
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    binding.uep_histogram_static(ids1, 256, out1)          # two calls in a row on one stream,
    binding.uep_histogram_static(ids2, 160, out2)          # no synchronisation between them
    binding.uep_histogram_static(ids1, 256, out3)          # and the first input again after the small one
    binding.uep_histogram_static(None, 16, empty)          # no slots at all: zeros
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0           # device memory in use did not move
    np.testing.assert_array_equal(out1.cpu().numpy(), want1)
    np.testing.assert_array_equal(out2.cpu().numpy(), want2)
    np.testing.assert_array_equal(out3.cpu().numpy(), want1)
    np.testing.assert_array_equal(empty.cpu().numpy(), np.zeros(16, np.int32))
    # and both against the oracle's definition (O-1), so that the two GPU paths cannot be wrong together
    np.testing.assert_array_equal(want1, oracle.histogram(ids1.cpu().numpy(), 256)[0])
    np.testing.assert_array_equal(out2.cpu().numpy(), oracle.histogram(ids2.cpu().numpy(), 160)[0])
    assert int(out2.sum().item()) == ids2.numel() - bad.numel()


@pytest.mark.gpu
def test_static_histogram_at_its_maximum_size():
    """Exactly UEP_STATIC_MAX_SLOTS slots (one more than a context accepts) against the oracle."""
    g = torch.Generator(device="cuda").manual_seed(4103)
    ids = torch.randint(-2, 514, (binding.STATIC_MAX_SLOTS,), generator=g, device="cuda", dtype=torch.int32)
    out = torch.full((512,), -7, dtype=torch.int32, device="cuda")
    binding.uep_histogram_static(ids, 512, out)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(out.cpu().numpy(), oracle.histogram(ids.cpu().numpy(), 512)[0])


def test_static_histogram_rejects_sizes_beyond_its_maximum():
    """Argument checks come before any CUDA call: they run without a GPU."""
    L = binding.lib()
    L.uep_histogram_static.restype = ctypes.c_int
    fake = ctypes.c_void_p(256)                            # aligned, never dereferenced: the call is rejected first

    def call(n, E, ids=fake, out=fake):
        return L.uep_histogram_static(ids, ctypes.c_longlong(n), ctypes.c_int32(E), out, ctypes.c_void_p(0))

    assert call(binding.STATIC_MAX_SLOTS + 1, 256) == -2
    msg = L.uep_static_last_error().decode()
    assert "UEP_STATIC_MAX_SLOTS" in msg and str(binding.STATIC_MAX_SLOTS + 1) in msg
    assert call(1024, 513) == -2 and "UEP_MAX_E" in L.uep_static_last_error().decode()
    assert call(1024, 0) == -2
    assert call(-1, 16) == -1
    assert call(1024, 16, out=ctypes.c_void_p(0)) == -1
    assert call(1024, 16, ids=ctypes.c_void_p(260)) == -1  # not 16-byte aligned
    with pytest.raises(binding.UepError, match="UEP_STATIC_MAX_SLOTS"):
        binding.uep_histogram_static(None, 16, None, stream=_NoStream(), n_slots=binding.STATIC_MAX_SLOTS + 1)


class _NoStream:
    cuda_stream = 0
