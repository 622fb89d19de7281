"""dimos_nl_needs_rebuild_static: the rebuild trigger (reading C-5) with its scratch in a fixed __device__
array, for callers that must not allocate.  Its flag must equal the flag of the existing path (dimos_nl_needs_rebuild)
and of the oracle on the same inputs, on two calls in a row (the array keeps the last call's contents); the reported
maximum squared displacement is compared with the oracle's within the rounding of the context's element type.  The call
must not touch the caller's allocator and must reject N beyond DIMOS_STATIC_MAX_ATOMS.

This file sorts last on purpose (pytest -x): it runs both alone and after the other GPU tests."""
import numpy as np
import pytest
import torch

import oracle
from paper_2503_20541_b200 import binding as dimos

pytestmark = pytest.mark.gpu

STATIC_MAX_ATOMS = 8388608  # include/dimos.h DIMOS_STATIC_MAX_ATOMS


def _case(n, seed, skin, scale, np_real):
    """Seeded positions whose displacements from the reference are uniform in [0, scale * skin / 2]."""
    rng = np.random.default_rng(seed)
    ref = rng.uniform(-3.0, 25.0, size=(n, 3)).astype(np_real)
    d = rng.normal(size=(n, 3))
    d *= (rng.uniform(0.0, 1.0, size=(n, 1)) * scale * 0.5 * skin) / np.linalg.norm(d, axis=1, keepdims=True)
    pos = (ref.astype(np.float64) + d).astype(np_real)
    return pos, ref


@pytest.mark.parametrize("precision", ["f32", "f64"])
@pytest.mark.parametrize("n", [1, 1000, 1024, 1025, 70001, 900000])
def test_static_trigger_matches_the_existing_path_twice_in_a_row(precision, n):
    np_real = np.float64 if precision == "f64" else np.float32
    rel = 1e-12 if precision == "f64" else 2e-6  # three squared differences of rounded coordinates of size <= 25
    dev = torch.device("cuda", 0)
    skin = 0.1
    ctx = dimos.Context(0, precision)
    try:
        flag_new = torch.full((1,), -7, dtype=torch.int32, device=dev)
        flag_old = torch.full((1,), -7, dtype=torch.int32, device=dev)
        m2 = torch.full((1,), -1.0, dtype=torch.float64, device=dev)
        # two calls in a row on different inputs: below the threshold, then above it (and back: the state left by a
        # call that fired must not leak into the next one)
        for rep, scale in enumerate((0.9, 1.6, 0.5)):
            pos_np, ref_np = _case(n, 100 * n + rep, skin, scale, np_real)
            pos, ref = torch.from_numpy(pos_np).to(dev), torch.from_numpy(ref_np).to(dev)
            dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, skin, flag_new, m2)
            dimos.dimos_nl_needs_rebuild(ctx, pos, ref, skin, sync=False, flag=flag_old)
            torch.cuda.synchronize()
            want, m = oracle.needs_rebuild(pos_np, ref_np, skin)
            got_new, got_old, got_m2 = int(flag_new.item()), int(flag_old.item()), float(m2.item())
            assert got_new in (0, 1)
            assert got_new == got_old, (rep, got_new, got_old)  # bit-exact against the existing path
            assert abs(got_m2 - m * m) <= rel * max(m * m, 1e-30) + 1e-300, (got_m2, m * m)
            if abs(m - 0.5 * skin) > 1e-6:  # away from the threshold the oracle decides, too
                assert bool(got_new) == want, (rep, m)
        # the same input twice in a row gives the same answer
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, skin, flag_new, m2)
        first = (int(flag_new.item()), float(m2.item()))
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, skin, flag_new, None)
        assert (int(flag_new.item()), float(m2.item())) == first
    finally:
        ctx.close()


def test_static_trigger_nan_forces_a_rebuild_and_strictness():
    dev = torch.device("cuda", 0)
    ctx = dimos.Context(0, "f32")
    try:
        flag = torch.zeros(1, dtype=torch.int32, device=dev)
        m2 = torch.zeros(1, dtype=torch.float64, device=dev)
        ref = torch.zeros(3000, 3, dtype=torch.float32, device=dev)
        pos = ref.clone()
        pos[1234, 1] = 0.25  # exactly skin/2 with skin = 0.5: strict >, no rebuild
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.5, flag, m2)
        assert int(flag.item()) == 0 and float(m2.item()) == 0.0625
        pos[1234, 1] = float(np.nextafter(np.float32(0.25), np.float32(1.0)))
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.5, flag, m2)
        assert int(flag.item()) == 1
        pos[1234, 1] = 0.0
        pos[2999, 2] = float("nan")
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.5, flag, m2)
        assert int(flag.item()) == 1 and float(m2.item()) == float("inf")
        pos[2999, 2] = 0.0
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.5, flag, m2)
        assert int(flag.item()) == 0 and float(m2.item()) == 0.0
    finally:
        ctx.close()


def test_static_trigger_allocates_nothing_and_rejects_sizes_beyond_its_array():
    dev = torch.device("cuda", 0)
    ctx = dimos.Context(0, "f32")
    try:
        n = 50000
        ref = torch.rand(n, 3, dtype=torch.float32, device=dev)
        pos = ref + 0.01
        flag = torch.zeros(1, dtype=torch.int32, device=dev)
        dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.1, flag)  # first call on the device: address look-up
        torch.cuda.synchronize()
        stats0 = torch.cuda.memory_stats(dev)
        free0, _ = torch.cuda.mem_get_info(dev)
        for _ in range(20):
            dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.1, flag)
        torch.cuda.synchronize()
        stats1 = torch.cuda.memory_stats(dev)
        free1, _ = torch.cuda.mem_get_info(dev)
        # the library's only route to device memory in this process is torch's caching allocator (binding.Context hands it
        # in as dimos_allocator) or cudaMalloc itself: neither moved
        assert stats1["allocation.all.allocated"] == stats0["allocation.all.allocated"]
        assert stats1["segment.all.allocated"] == stats0["segment.all.allocated"]
        assert free1 == free0
        assert int(flag.item()) == 0
        # sizes beyond the array: clear error, nothing launched, flag untouched.  The call reads only N before it refuses,
        # so small tensors can stand in for the 8 M-atom arrays.
        flag.fill_(-3)
        launches = ctx.launch_count()
        rc = ctx.lib.dimos_nl_needs_rebuild_static(ctx.handle, pos.data_ptr(), ref.data_ptr(), STATIC_MAX_ATOMS + 1, 0.1,
                                                   flag.data_ptr(), None, None)
        assert rc == -4  # DIMOS_EOVERFLOW
        assert "DIMOS_STATIC_MAX_ATOMS" in ctx.lib.dimos_last_error(ctx.handle).decode()
        assert ctx.launch_count() == launches
        torch.cuda.synchronize()
        assert int(flag.item()) == -3
    finally:
        ctx.close()


def test_static_trigger_at_its_maximum_size_f32():
    """N = DIMOS_STATIC_MAX_ATOMS: every block-maximum slot of the array is in use; the one displaced atom sits in the last
    block.  Compared with the existing path (bit-exact) and the oracle."""
    dev = torch.device("cuda", 0)
    n = STATIC_MAX_ATOMS
    ctx = dimos.Context(0, "f32")
    try:
        rng = np.random.default_rng(5)
        ref_np = rng.uniform(0.0, 40.0, size=(n, 3)).astype(np.float32)
        pos_np = ref_np.copy()
        flag_new = torch.zeros(1, dtype=torch.int32, device=dev)
        flag_old = torch.zeros(1, dtype=torch.int32, device=dev)
        m2 = torch.zeros(1, dtype=torch.float64, device=dev)
        ref = torch.from_numpy(ref_np).to(dev)
        for shift in (0.03, 0.07):  # below, then above skin / 2 = 0.05
            pos_np[n - 1, 0] = ref_np[n - 1, 0] + np.float32(shift)
            pos = torch.from_numpy(pos_np).to(dev)
            dimos.dimos_nl_needs_rebuild_static(ctx, pos, ref, 0.1, flag_new, m2)
            dimos.dimos_nl_needs_rebuild(ctx, pos, ref, 0.1, sync=False, flag=flag_old)
            torch.cuda.synchronize()
            want, m = oracle.needs_rebuild(pos_np, ref_np, 0.1)
            assert int(flag_new.item()) == int(flag_old.item()) == int(want)
            assert abs(float(m2.item()) - m * m) <= 2e-6 * m * m
    finally:
        ctx.close()
