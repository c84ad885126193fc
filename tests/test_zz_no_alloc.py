"""ks_depth_bound_static -- the one entry point of the library whose kernel works in memory that is
part of the library image instead of memory the caller lends (include/kineticsim.h).

It is there for callers who cannot allocate device memory at the moment they want to vet a book
image: a thread next to a running simulation (cudaMalloc / cudaFree wait for the device, i.e. for a
ks_run that may hold it for hundreds of milliseconds), a process whose framework pool already owns
all of HBM (cudaMalloc fails), or code under a no-allocation-after-start-up rule.  The usual depth
check (behind ks_write_books / ks_attach) borrows a word from the tail of the caller's d_state; such
a caller has no d_state yet.

The GPU test compares the new call with that existing path -- the word ks_write_books' check leaves
in the library-scratch tail of d_state -- and with the plain definition in numpy, bit for bit (it is
integer work), on two calls in a row that share the library's array: the second image is smaller in
every way, so a result that leaked from the first call's leftovers would be too large.

This file is named to be collected last: under `pytest -x` a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call on the device does the address
look-up) and after the other tests.
"""

import numpy as np
import pytest

from paper_2606_21784_b200 import binding, build
from paper_2606_21784_b200.workloads import zi_params

ALL_ONES = 0xFFFFFFFFFFFFFFFF


def _definition(books: np.ndarray) -> int:
    """max over markets and sides of the per-side total; all ones if any entry is negative."""
    if (books < 0).any():
        return ALL_ONES
    return int(books.astype(np.int64).sum(axis=2).max())


def test_static_depth_bound_rejects_bad_sizes_before_touching_cuda():
    """Argument checks come first, so they are testable without a GPU: beyond the limit the call
    says what the limit is and why, and enqueues nothing."""
    build.build()
    lib = binding.load()
    dummy_in = np.zeros(64, dtype=np.int32)
    dummy_out = np.zeros(1, dtype=np.uint64)
    too_many = binding.KS_DEPTH_BOUND_STATIC_MAX_M + 1
    assert lib.ks_depth_bound_static(dummy_in.ctypes.data, too_many, 32, dummy_out.ctypes.data, None) == binding.KS_ERR_UNSUPPORTED
    text = binding.ks_last_error()
    assert "KS_DEPTH_BOUND_STATIC_MAX_M = 65536" in text and str(too_many) in text
    for (M, L) in ((0, 32), (1, 48), (1, 16), (1, 65536)):
        assert lib.ks_depth_bound_static(dummy_in.ctypes.data, M, L, dummy_out.ctypes.data, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_depth_bound_static(None, 1, 32, dummy_out.ctypes.data, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_depth_bound_static(dummy_in.ctypes.data, 1, 32, None, None) == binding.KS_ERR_INVALID_ARG
    assert lib.ks_depth_bound_static(dummy_in.ctypes.data, 1, 32, dummy_out.ctypes.data + 4, None) == binding.KS_ERR_INVALID_ARG
    # the header's constant and the binding's agree
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    hdr = open(os.path.join(root, "include", "kineticsim.h")).read()
    assert int(re.search(r"#define\s+KS_DEPTH_BOUND_STATIC_MAX_M\s+(\d+)", hdr).group(1)) == binding.KS_DEPTH_BOUND_STATIC_MAX_M


def test_static_entry_point_allocates_nothing_in_source():
    """The promise is checkable in the source: no allocating CUDA call anywhere in the translation unit
    except the handle's pinned words in ks_create (cudaHostAlloc), which this entry point never reaches."""
    import os
    import re
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = open(os.path.join(root, "paper_2606_21784_b200", "csrc", "ks_api.cu")).read()
    body = src[src.index("static __device__ __align__(256) unsigned long long g_static_scratch"):]
    assert not re.search(r"\bcuda(Malloc\w*|Free\w*|HostAlloc|HostRegister|MemPool\w*|StreamCreate\w*|EventCreate\w*)\s*\(", body)
    assert "cudaGetSymbolAddress((void**)&ptr, g_static_scratch)" in body


def _existing_path(torch, books_host: np.ndarray, M: int, L: int) -> int:
    """The depth check the library already had: ks_write_books on a real d_state leaves its result
    in the first word of the 256-byte library-scratch tail of that buffer."""
    sim = binding.KsSim(M, L, 32, zi_params(4, 10), 1)
    src = torch.from_numpy(books_host).cuda()
    sim.ks_write_books(src)
    torch.cuda.current_stream().synchronize()
    off = M * (8 * L + 128)
    word = sim.state[off:off + 8].cpu().numpy().view(np.uint64)[0]
    sim.ks_destroy()
    return int(word)


@pytest.mark.gpu
def test_static_depth_bound_matches_the_existing_check_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available()
    build.build()
    binding.load()
    rng = np.random.default_rng(20261106)
    # call 1: many markets, deep books (ragged grid: 2*301 blocks); call 2: few markets, shallow books,
    # another L -- everything the first call left in the library's array is larger than the right answer
    first = rng.integers(0, 50000, size=(301, 2, 512), dtype=np.int32)
    second = rng.integers(0, 7, size=(5, 2, 64), dtype=np.int32)
    third = second.copy()
    third[3, 1, 17] = -1                                    # a negative entry anywhere -> all ones
    images = [first, second, third, first]
    want_existing = [_existing_path(torch, b, b.shape[0], b.shape[2]) for b in images]
    want_definition = [_definition(b) for b in images]
    assert want_existing == want_definition                 # the two references agree with each other
    assert want_definition[1] < want_definition[0] and want_definition[2] == ALL_ONES

    d_books = [torch.from_numpy(b).cuda() for b in images]
    d_out = torch.zeros(len(images), dtype=torch.int64, device="cuda")
    # the first call on this device (when this file runs alone): the library looks up its array's
    # address and the runtime loads the kernel; its result counts like any other
    binding.ks_depth_bound_static(d_books[1], 5, 64, d_out[3:4])
    torch.cuda.synchronize()
    assert int(d_out[3].item()) == want_definition[1]
    before = binding.ks_launch_count()
    mem_before = torch.cuda.mem_get_info()[0]
    # back to back on ONE stream, no synchronisation in between: the calls share the library's array
    for i, b in enumerate(images):
        binding.ks_depth_bound_static(d_books[i], b.shape[0], b.shape[2], d_out[i:i + 1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == mem_before       # the driver handed out no device memory
    assert binding.ks_launch_count() - before == len(images)  # one kernel per call
    got = [int(x) for x in d_out.cpu().numpy().view(np.uint64)]
    assert got == want_existing                             # integer work: bit-exact, as in the parity tests

    # at the limit itself the call is accepted (M = KS_DEPTH_BOUND_STATIC_MAX_M, smallest L)
    Mmax = binding.KS_DEPTH_BOUND_STATIC_MAX_M
    big = torch.ones((Mmax, 2, 32), dtype=torch.int32, device="cuda")
    big[Mmax - 1, 0, :] = 3
    binding.ks_depth_bound_static(big, Mmax, 32, d_out[0:1])
    torch.cuda.synchronize()
    assert int(d_out[0].item()) == 96
    with pytest.raises(binding.KsError) as err:
        binding.ks_depth_bound_static(big, Mmax + 1, 32, d_out[0:1])
    assert err.value.status == binding.KS_ERR_UNSUPPORTED
