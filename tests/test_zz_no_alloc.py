"""GPU test of sph_select_range_static (include/sph.h): the selection kernels of sph_select_range with their flag / scan
scratch in a file-scope `static __device__` array of the library instead of caller memory -- the entry point for callers
that cannot call cudaMalloc.  Its output must equal the existing path's bit for bit (integer and copy work), on two
calls in a row (the second one smaller, so that it runs on the first one's stale scratch), at the maximum size, and
sizes beyond the maximum must be rejected with a clear error.

Collected last on purpose (file name): the suite runs with `pytest -x`."""
import ctypes as C

import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device")
    from paper_2403_11156_b200 import binding, build
    build.build()
    binding.load()
    return binding


STATIC_MAX = 1 << 20        # SPH_SELECT_STATIC_MAX of include/sph.h


def _case(torch, n, seed, with_key):
    """Seeded synthetic input of a slab selection: positions in a 4 m tank, ids a permutation, key = original index of
    the slot (slab mode: < key_lt means owned)."""
    g = torch.Generator().manual_seed(seed)
    pos = torch.rand((n, 4), generator=g, dtype=torch.float32)
    pos[:, 0] *= 4.0
    vel = torch.rand((n, 4), generator=g, dtype=torch.float32) - 0.5
    gid = torch.randperm(n, generator=g).to(torch.int32)
    key = torch.randperm(n, generator=g).to(torch.int32) if with_key else None
    d = lambda t: t.cuda() if t is not None else None
    return d(pos), d(vel), d(gid), d(key)


def _run(B, torch, stream, static, pos, vel, gid, key, key_lt, lo, hi, max_out, want_idx):
    n = pos.shape[0]
    dev = pos.device
    opos = torch.full((max(max_out, 1), 4), -7.0, dtype=torch.float32, device=dev)
    ovel = torch.full((max(max_out, 1), 4), -7.0, dtype=torch.float32, device=dev)
    ogid = torch.full((max(max_out, 1),), -7, dtype=torch.int32, device=dev)
    oidx = torch.full((max(max_out, 1),), -7, dtype=torch.int32, device=dev) if want_idx else None
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    cnt = C.c_int(-1)
    L = B.load()
    torch.cuda.synchronize()
    if static:
        rc = L.sph_select_range_static(C.c_void_p(stream.cuda_stream), p(pos), p(vel), p(gid), p(key), int(key_lt), n,
                                       float(lo), float(hi), p(opos), p(ovel), p(ogid), p(oidx), int(max_out), C.byref(cnt))
    else:
        scratch = torch.full((n + 8 + (n + 1) // 4096 + 8,), 0x5a5a5a5a, dtype=torch.int32, device=dev)
        torch.cuda.synchronize()
        rc = L.sph_select_range(C.c_void_p(stream.cuda_stream), p(pos), p(vel), p(gid), p(key), int(key_lt), n,
                                float(lo), float(hi), p(opos), p(ovel), p(ogid), p(oidx), int(max_out),
                                p(scratch), scratch.numel(), C.byref(cnt))
    assert rc == B.SPH_OK, (rc, L.sph_last_error(None))
    torch.cuda.synchronize()
    return cnt.value, opos, ovel, ogid, oidx


def _check_pair(B, torch, stream, n, seed, with_key, lo, hi, max_out=None):
    pos, vel, gid, key = _case(torch, n, seed, with_key)
    key_lt = (2 * n) // 3
    max_out = n if max_out is None else max_out
    ref = _run(B, torch, stream, False, pos, vel, gid, key, key_lt, lo, hi, max_out, True)
    new = _run(B, torch, stream, True, pos, vel, gid, key, key_lt, lo, hi, max_out, True)
    assert new[0] == ref[0]
    for a, b in zip(new[1:], ref[1:]):
        assert torch.equal(a, b)                      # bit-exact, the untouched tail (-7) included
    # and both equal the plain definition: input order kept, x in [lo, hi), key < key_lt
    m = (pos[:, 0] >= lo) & (pos[:, 0] < hi)
    if key is not None:
        m &= key < key_lt
    idx = torch.nonzero(m).flatten()
    assert new[0] == idx.numel()
    k = min(idx.numel(), max_out)
    assert torch.equal(new[4][:k].long(), idx[:k])
    assert torch.equal(new[1][:k], pos[idx[:k]]) and torch.equal(new[2][:k], vel[idx[:k]])
    src = key[idx[:k]].long() if key is not None else idx[:k]
    assert torch.equal(new[3][:k], gid[src])
    return new[0]


def test_static_scratch_selection_equals_caller_scratch_selection(B):
    import torch
    stream = torch.cuda.Stream()
    # two calls in a row: several scan tiles + a ragged tail, then a smaller call on the stale scratch of the first
    c1 = _check_pair(B, torch, stream, 300_017, 1, True, 1.0, 2.4)
    c2 = _check_pair(B, torch, stream, 70_001, 2, False, 0.5, 3.5)
    assert c1 > 10_000 and c2 > 10_000
    # the first call again: identical to itself whatever the scratch held in between; output buffer smaller than the
    # selection (the count is still the full one); empty selection; a single entry
    assert _check_pair(B, torch, stream, 300_017, 1, True, 1.0, 2.4) == c1
    assert _check_pair(B, torch, stream, 50_000, 3, True, 0.0, 4.0, max_out=1000) > 1000
    assert _check_pair(B, torch, stream, 4097, 4, False, 5.0, 6.0) == 0
    assert _check_pair(B, torch, stream, 1, 5, False, 0.0, 4.0) == 1


def test_static_scratch_maximum_size_and_rejection_beyond_it(B):
    import torch
    stream = torch.cuda.Stream()
    assert _check_pair(B, torch, stream, STATIC_MAX, 6, True, 0.0, 2.0) > 100_000
    L = B.load()
    cnt = C.c_int(5)
    rc = L.sph_select_range_static(C.c_void_p(stream.cuda_stream), None, None, None, None, 0, STATIC_MAX + 1, 0.0, 1.0,
                                   None, None, None, None, 0, C.byref(cnt))
    assert rc == B.SPH_EINVAL and cnt.value == 0
    msg = (L.sph_last_error(None) or b"").decode()
    assert "SPH_SELECT_STATIC_MAX" in msg and str(STATIC_MAX) in msg, msg
    assert L.sph_select_range_static(None, None, None, None, None, 0, 5, 0.0, 1.0, None, None, None, None, 0, None) == B.SPH_EINVAL
    # n = 0 is valid and selects nothing
    cnt = C.c_int(5)
    assert L.sph_select_range_static(C.c_void_p(stream.cuda_stream), None, None, None, None, 0, 0, 0.0, 1.0,
                                     None, None, None, None, 0, C.byref(cnt)) == B.SPH_OK and cnt.value == 0


def test_static_scratch_call_allocates_no_device_memory(B):
    """Free device memory as the driver reports it does not move across calls of the entry point (inputs and outputs
    are allocated before; the first call of a process may load the module lazily, so it is not the one measured)."""
    import torch
    stream = torch.cuda.Stream()
    pos, vel, gid, key = _case(torch, 200_003, 7, True)
    first = _run(B, torch, stream, True, pos, vel, gid, key, 100_000, 1.0, 3.0, 200_003, True)
    dev = pos.device
    opos = torch.empty((200_003, 4), dtype=torch.float32, device=dev)
    ovel = torch.empty((200_003, 4), dtype=torch.float32, device=dev)
    ogid = torch.empty((200_003,), dtype=torch.int32, device=dev)
    p = lambda t: C.c_void_p(t.data_ptr())
    L = B.load()
    cnt = C.c_int(-1)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        rc = L.sph_select_range_static(C.c_void_p(stream.cuda_stream), p(pos), p(vel), p(gid), p(key), 100_000, 200_003,
                                       1.0, 3.0, p(opos), p(ovel), p(ogid), None, 200_003, C.byref(cnt))
        assert rc == B.SPH_OK and cnt.value == first[0]
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert torch.equal(opos[:cnt.value], first[1][:cnt.value]) and torch.equal(ogid[:cnt.value], first[3][:cnt.value])
