"""ddf_gen_shadow_from_hits_static: the shadow-ray compaction for programs that cannot allocate device memory.

Who needs it: a host that handed the whole GPU to its own memory pool at start-up (a renderer with a fixed budget, a
framework's caching allocator), so that a cudaMalloc made on the library's behalf fails; or a frame loop that cannot
take the device-wide stall of cudaMalloc / cudaFree.  ddf_gen_shadow_from_hits keeps the block counts of its stable
compaction in a cudaMalloc'ed workspace owned by a model; the _static variant keeps them in a fixed 256 KB array
inside libddf.so, takes no model, and is limited to 2^24 rays (include/ddf.h).

What is checked: on two calls in a row (the second smaller, with other data and another light, so that anything the
first left in the shared array would show) the _static entry point returns exactly what the model-owned path returns -
the two launch the same kernels, so the tolerance is zero, the tightest the wavefront tests use (indices bit-exact);
the free device memory is the same before and after a call; a batch over the limit is refused with its own status.
This file sorts last on purpose (pytest -x stops at the first failure), and passes alone in a fresh process as well as
after the rest of the suite: it builds its own model and inputs and depends on no state another test leaves behind.
"""
import ctypes as C

import numpy as np
import pytest


def _libddf():
    from paper_2606_00817_b200 import build, lib
    build()
    return lib()


def test_static_entry_point_refuses_oversized_and_negative_batches_without_a_gpu():
    lib = _libddf()
    li = (C.c_float * 3)(1.0, 2.0, 3.0)
    cnt = C.c_int64(0)                                  # never dereferenced: both calls return before any CUDA work
    args = (None, None, None, None)
    assert lib.ddf_gen_shadow_from_hits_static(*args, C.c_int64((1 << 24) + 1), li, C.c_float(1e-3), None, None, None, None, C.byref(cnt), None) == -6
    assert lib.ddf_gen_shadow_from_hits_static(*args, C.c_int64(-1), li, C.c_float(1e-3), None, None, None, None, C.byref(cnt), None) == -1
    assert lib.ddf_gen_shadow_from_hits_static(*args, C.c_int64(4), None, C.c_float(1e-3), None, None, None, None, C.byref(cnt), None) == -1
    from paper_2606_00817_b200 import ddf_status_string, STATIC_MAX_RAYS
    assert "capacity" in ddf_status_string(-6) and STATIC_MAX_RAYS == 1 << 24


@pytest.mark.gpu
def test_static_entry_point_matches_the_model_owned_path_on_two_calls_in_a_row():
    import torch
    import paper_2606_00817_b200 as ddf
    from ddf_inputs import layout_c0, make_weights, random_rays
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    lay = layout_c0()
    m = ddf.ddf_create(make_weights(lay), lay)

    def primary(n, seed):
        o, d = random_rays(n, seed=seed)
        o, d = torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda()
        dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
        ddf.ddf_query(m, o, d, n, dist, vis)
        return o, d, dist, vis

    def outputs(n):
        return (torch.full((n, 3), 7.0, device="cuda"), torch.full((n, 3), 7.0, device="cuda"), torch.full((n,), 7.0, device="cuda"),
                torch.full((n,), -1, dtype=torch.int32, device="cuda"), torch.full((1,), -1, dtype=torch.int64, device="cuda"))

    # 391 count blocks with a ragged tail, then 79: the second call reads a strict prefix of what the first wrote
    cases = [(100_003, 11, (3.0, 3.0, 3.0), 1e-3), (20_011, 12, (-2.0, 0.5, 4.0), 1e-2)]
    batches = [primary(n, seed) for n, seed, _, _ in cases]
    want = []
    for (n, _, light, eps), (o, d, dist, vis) in zip(cases, batches):
        ref = outputs(n)
        ddf.ddf_gen_shadow_from_hits(m, o, d, dist, vis, n, light, eps, *ref)
        want.append(ref)
    # start-up call on this device (looks the array's address up), as the header asks for
    warm = outputs(cases[1][0])
    ddf.ddf_gen_shadow_from_hits_static(*batches[1], cases[1][0], cases[1][2], cases[1][3], *warm)
    torch.cuda.synchronize()
    got = [outputs(n) for n, _, _, _ in cases]
    free_before = torch.cuda.mem_get_info()[0]
    for (n, _, light, eps), (o, d, dist, vis), out in zip(cases, batches, got):          # two calls in a row, one stream
        ddf.ddf_gen_shadow_from_hits_static(o, d, dist, vis, n, light, eps, *out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the static entry point must not allocate device memory"
    for (n, _, _, _), (_, _, _, vis), ref, out in zip(cases, batches, want, got):
        k = int(ref[4].item())
        assert k == int((vis > 0.5).sum().item()) and 0 < k < n, (n, k)
        assert int(out[4].item()) == k
        assert torch.equal(out[3][:k], ref[3][:k])                                     # index: which primary ray
        assert bool((out[3][:k][1:] > out[3][:k][:-1]).all())                          # stable: increasing
        for a, b in zip(out[:3], ref[:3]):                                             # o2, d2, tmax: same kernels, same bits
            assert torch.equal(a[:k], b[:k])
            assert torch.equal(a[k:], torch.full_like(a[k:], 7.0))                     # nothing written past the count
    # the warm-up call saw the second batch as well
    k = int(want[1][4].item())
    assert int(warm[4].item()) == k and torch.equal(warm[3][:k], want[1][3][:k])
    # an empty batch reports zero rays; a batch over the limit is refused by name
    cnt = torch.full((1,), 5, dtype=torch.int64, device="cuda")
    ddf.ddf_gen_shadow_from_hits_static(None, None, None, None, 0, (0.0, 0.0, 1.0), 1e-3, None, None, None, None, cnt)
    assert int(cnt.item()) == 0
    with pytest.raises(ddf.DdfError, match="capacity"):
        ddf.ddf_gen_shadow_from_hits_static(*batches[0], ddf.STATIC_MAX_RAYS + 1, (0.0, 0.0, 1.0), 1e-3, *got[0])
    ddf.ddf_destroy(m)
