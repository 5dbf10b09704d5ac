"""dwf_norm2_static: the entry point for callers that cannot let this library allocate device memory.

Who that is: applications that took the whole GPU into their own memory pool at start-up (lattice codes and tensor
frameworks do, so a cudaMalloc from inside a library fails or cuts into their pool), latency-critical code that cannot take
the device-wide synchronisation a cudaMalloc / cudaFree implies, and plug-ins whose host forbids allocating in callbacks.
For them the per-block partial sums of the norm live in a fixed 512 KiB array built into libdwf_b200.so instead of the
cudaMalloc'ed buffer a dwf context owns; the price is an input limit of 4 GiB (include/dwf.h, DWF_NORM2_STATIC_MAX_BYTES).

What is checked: on the GPU, that the new entry point gives what the existing dwf_norm2 gives, to the 1e-13 / 1e-12 relative
bars tests/test_gpu_parity.py::test_norm2_and_convert uses for that routine, on two calls in a row that share the array
(a large field first, a smaller one second, so that leftovers of the first call would show); on any box, that an input over
the limit is refused with a message and that nothing is launched for it.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests of the hot path.  It passes run alone in a fresh process (where its first call is the one that looks up the
array's address) and after the rest of the suite.
"""
import ctypes

import pytest

from paper_2203_17119_b200 import api


def _call(lib, ptr, nreal, prec, out_ptr=0x1000, stream=None):
    err = ctypes.create_string_buffer(256)
    st = lib.dwf_norm2_static(ctypes.c_void_p(ptr), nreal, prec, ctypes.c_void_p(out_ptr), ctypes.c_void_p(stream), err, len(err))
    return st, err.value.decode()


def test_static_norm_refuses_what_its_fixed_scratch_cannot_serve():
    """Argument checks come before any CUDA call, so they run on the CPU-only box too: the pointers below are never
    dereferenced.  One real over the 4 GiB limit is too many; the message names the limit."""
    lib = api.load_library()
    assert api.NORM2_STATIC_MAX_BYTES == 1 << 32
    for prec, size in ((api.F64, 8), (api.F32, 4)):
        over = api.NORM2_STATIC_MAX_BYTES // size + 16 // size
        st, msg = _call(lib, 0x10000, over, prec)
        assert st == api.EINVAL and "DWF_NORM2_STATIC_MAX_BYTES" in msg and str(api.NORM2_STATIC_MAX_BYTES) in msg, msg
    st, msg = _call(lib, 0x10000, 2 ** 63, api.F64)                       # no overflow in the size arithmetic
    assert st == api.EINVAL and "DWF_NORM2_STATIC_MAX_BYTES" in msg
    st, msg = _call(lib, 0x10008, 64, api.F64)
    assert st == api.EINVAL and "aligned" in msg
    st, msg = _call(lib, 0, 64, api.F64)
    assert st == api.EINVAL and "null" in msg
    st, msg = _call(lib, 0x10000, 64, api.F64, out_ptr=0)
    assert st == api.EINVAL and "result_dev" in msg
    st, msg = _call(lib, 0x10000, 63, api.F64)
    assert st == api.EINVAL and "16-byte vectors" in msg
    st, msg = _call(lib, 0x10000, 64, 7)
    assert st == api.EINVAL and "prec" in msg
    # a null message buffer is allowed
    assert lib.dwf_norm2_static(ctypes.c_void_p(0), 64, api.F64, ctypes.c_void_p(0x1000), None, None, 0) == api.EINVAL


@pytest.mark.gpu
def test_static_norm_matches_dwf_norm2_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available()
    dev = torch.device("cuda:0")
    gen = torch.Generator(device=dev).manual_seed(20220317)
    big = api.Dwf((8, 8, 8, 8), 8, 1.8, 0.01, 1.5, 0.5)                   # 196608 fp64 vectors: 48 full blocks
    small = api.Dwf((4, 4, 4, 4), 3, 1.8, 0.01, 1.0, 0.0)                 # 4608 vectors: one full block and a ragged one
    out = torch.full((2,), float("nan"), dtype=torch.float64, device=dev)  # the caller's output, one slot per call
    try:
        for prec, bar in ((api.F64, 1e-13), (api.F32, 1e-12)):
            # values of very different size in the two fields: partial sums left behind by the first call (~1e6 each)
            # would swamp the second result (~1e-2) if they were ever read
            a = big.new_native(prec, api.ODD).normal_(generator=gen).mul_(30.0)
            b = small.new_native(prec, api.ODD).normal_(generator=gen).mul_(1e-3)
            want_a, want_b = big.norm2(a, prec, api.ODD), small.norm2(b, prec, api.ODD)     # the existing path
            out.fill_(float("nan"))
            api.norm2_static(a, out[0:1])                                  # two calls back to back on one stream,
            api.norm2_static(b, out[1:2])                                  # nothing in between
            got_a, got_b = out.tolist()
            assert abs(got_a - want_a) <= bar * want_a, (prec, got_a, want_a)
            assert abs(got_b - want_b) <= bar * want_b, (prec, got_b, want_b)
            assert want_a > 1e6 * want_b > 0.0
            # and a third time on the first field: the same bits as before (fixed summation tree)
            again = torch.zeros(1, dtype=torch.float64, device=dev)
            api.norm2_static(a, again)
            assert again.item() == got_a
        # an empty input is a sum over nothing; a FULL field (two halves back to back) is just a longer array
        api.norm2_static(torch.empty(0, dtype=torch.float64, device=dev), out[0:1])
        assert out[0].item() == 0.0
        f = big.new_native(api.F64, api.FULL).normal_(generator=gen)
        api.norm2_static(f, out[1:2])
        want = big.norm2(f, api.F64, api.FULL)
        assert abs(out[1].item() - want) <= 1e-13 * want
        # over the limit: refused with DwfError before anything is enqueued (the tensor's size is faked through the ABI)
        st, msg = _call(api.load_library(), a.data_ptr(), api.NORM2_STATIC_MAX_BYTES // 4 + 4, api.F32, out.data_ptr(),
                        torch.cuda.current_stream(dev).cuda_stream)
        assert st == api.EINVAL and "DWF_NORM2_STATIC_MAX_BYTES" in msg
        torch.cuda.synchronize(dev)
    finally:
        big.close()
        small.close()
