"""sph_sort_keys_static: the neighbour-list sort for callers that cannot allocate device memory.

Some users of this library sit inside a host program that has taken the whole GPU into its own memory pool (a coupled
solver with a fixed budget, a plug-in with no allocator callback to hand to sph_create), or inside a loop that must not
take the device-wide stall of cudaMalloc / cudaFree.  For them the library offers one call that allocates nothing: the
radix sort of the cell keys, run on a work space compiled into the library (a static __device__ array, about 8.3 MiB per
GPU, at most SPH_SORT_STATIC_MAX_N = 2^20 keys).

What is checked here: the call gives exactly the sorted keys and the permutation of the ordinary context path
(sph_load_particles + sph_compute_interactions, SPH_KEY / SPH_PERM) -- integer work, so the tolerance is bit equality,
as in test_gpu_parity.py -- on several calls in a row with different sizes and pass counts, because every call reuses
the same work space and finds the previous call's leftovers in it.  The free device memory must not move across the
calls.  This file is named so that pytest collects it last: with `pytest -x` a failure here hides no other test.  It
passes alone in a fresh process (the first call then does the per-device address look-up) and after the other files.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2104_00537_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sph():
    from paper_2104_00537_b200 import build
    build.build()
    from paper_2104_00537_b200 import sph as mod
    return mod


def test_size_limit_is_rejected_with_a_message(sph):
    """Too many keys for the built-in work space: SPH_E_OVERFLOW and a message that names the limit, decided before
    any CUDA call is made (so this runs on a box without a GPU too).  n = 0 is a no-op."""
    hdr = open(os.path.join(ROOT, "include", "sph.h")).read()
    assert int(re.search(r"#define\s+SPH_SORT_STATIC_MAX_N\s+(\d+)", hdr).group(1)) == sph.SPH_SORT_STATIC_MAX_N
    msg = C.create_string_buffer(512)
    rc = sph.lib.sph_sort_keys_static(None, sph.SPH_SORT_STATIC_MAX_N + 1, 24, None, None, None, msg, len(msg))
    assert rc == sph.SPH_E_OVERFLOW
    assert b"SPH_SORT_STATIC_MAX_N" in msg.value and str(sph.SPH_SORT_STATIC_MAX_N).encode() in msg.value
    with pytest.raises(sph.SphError, match="SPH_E_OVERFLOW"):
        sph.sort_keys_static(None, sph.SPH_SORT_STATIC_MAX_N + 1, 24, None, None)
    assert sph.lib.sph_sort_keys_static(None, 0, 24, None, None, None, None, 0) == sph.SPH_OK
    assert sph.lib.sph_sort_keys_static(None, -1, 24, None, None, None, msg, len(msg)) == sph.SPH_E_BADARG
    assert sph.lib.sph_sort_keys_static(None, 8, 0, None, None, None, msg, len(msg)) == sph.SPH_E_BADARG
    assert sph.lib.sph_sort_keys_static(None, 8, 24, None, None, None, msg, len(msg)) == sph.SPH_E_BADARG
    assert b"null" in msg.value


def _context_path(sph, case):
    """The existing path: first neighbour-list build after a load.  Returns (keys in load order, sorted keys,
    permutation, key_bits the context used).  After the first build the particles were still in load order when they
    were sorted, so SPH_PERM is the sort's own permutation and the unsorted keys follow by scattering the sorted ones
    back -- no key arithmetic is repeated here."""
    with sph.Sph(case.params) as S:
        S.load_case(case)
        S.compute_interactions()
        key_sorted = S.read_state(sph.SPH_KEY)
        perm = S.read_state(sph.SPH_PERM)
        info = S.get_info()
    key = np.empty_like(key_sorted)
    key[perm] = key_sorted
    return key, key_sorted, perm, int(2 * info.ncells).bit_length()


@pytest.mark.gpu
def test_static_sort_equals_the_context_path_on_calls_in_a_row(sph):
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    torch.cuda.set_device(0)
    # A: as many keys as the work space takes (256 blocks), fluid + boundary + a few out-of-grid particles, 3 passes.
    # B: a small shuffled dam break (5 blocks, ragged tail), sorted over all 32 bits (4 passes: the other ping-pong
    #    parity), right after A, so most of the work space still holds A's data.
    big = wl.random_cloud("static_a", sph.SPH_SORT_STATIC_MAX_N, (1.6, 1.6, 1.6), 0.01, 4242)
    big.pos[:7, 2] += 5.0                     # out of the grid: key 2 * ncells, sorted last
    small = wl.dam_break("static_b", 3, 0.02, (50, 25, 25), (15, 25, 15), 0.01, 99, 0.3, shuffle=True)
    refs = {"A": _context_path(sph, big), "B": _context_path(sph, small)}
    assert refs["A"][0].size == sph.SPH_SORT_STATIC_MAX_N and refs["A"][3] <= 24 < 32

    stream = torch.cuda.current_stream()
    dev = {}
    for name, (key, _, _, _) in refs.items():        # every buffer exists before the first call
        n = key.size
        dev[name] = (torch.from_numpy(key.view(np.int32)).cuda(), torch.empty(n, dtype=torch.int32, device="cuda"),
                     torch.empty(n, dtype=torch.int32, device="cuda"))
    torch.cuda.synchronize()

    def run(name, key_bits):
        k, ks, pm = dev[name]
        ks.fill_(-1)
        pm.fill_(-1)
        sph.sort_keys_static(k.data_ptr(), k.numel(), key_bits, ks.data_ptr(), pm.data_ptr(), stream.cuda_stream)
        got_keys = ks.cpu().numpy().view(np.uint32)
        got_perm = pm.cpu().numpy().view(np.uint32)
        key, key_sorted, perm, _ = refs[name]
        assert np.array_equal(k.cpu().numpy().view(np.uint32), key), f"{name}: the input keys were modified"
        assert np.array_equal(got_keys, key_sorted), f"{name}: sorted keys differ from the context path"
        assert np.array_equal(got_perm, perm), f"{name}: permutation differs from the context path"

    run("A", refs["A"][3])                    # first call: may include the one-off address look-up
    free0 = torch.cuda.mem_get_info()[0]
    run("B", 32)                              # second call in a row, different size and pass count
    run("A", refs["A"][3])                    # and back: B's leftovers are in the work space now
    run("B", refs["B"][3])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory was allocated or released during the calls"

    with pytest.raises(sph.SphError, match="three different arrays"):
        k, ks, _ = dev["B"]
        sph.sort_keys_static(k.data_ptr(), k.numel(), 24, ks.data_ptr(), ks.data_ptr(), stream.cuda_stream)
