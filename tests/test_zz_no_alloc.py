"""psg_range_rgyr_static (include/psg_static.h): the one entry point that allocates nothing (scratch in a static device
array) against the existing path, psg_cv_eval on a context, on the same inputs; two calls in a row share the scratch.

Collected last on purpose (the file name): the suite runs with `pytest -x`, a failure here must hide nothing.
Tolerance: the one of every CV comparison in tests/ (BASELINE.json north_star: 1e-5 relative, 1e-6 absolute floor)."""
import ctypes

import numpy as np
import pytest

from _parity import ABS, REL, assert_close

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def psg():
    import paper_2301_04835_b200 as p
    p.load_library()      # fails loudly if libpsg.so is missing: no fallback
    return p


def _positions(seed, R, N, ps):
    """a random-walk chain per replica (bond length 1) plus a replica-dependent offset: Rg ~ sqrt(N/6), far from the origin"""
    rng = np.random.default_rng(seed)
    steps = rng.normal(size=(R, N, 3))
    steps /= np.linalg.norm(steps, axis=2, keepdims=True)
    xyz = np.cumsum(steps, axis=1) + rng.uniform(-50, 50, size=(R, 1, 3))
    pos = np.zeros((R, N, ps), np.float32)
    pos[..., :3] = xyz
    if ps == 4:
        pos[..., 3] = rng.uniform(-1, 1, size=(R, N))      # the 4th float is ignored by both paths
    return pos


def _existing_path(torch, psg, pos, first, count, weight):
    """psg_cv_eval on a context: Rg and the three barycenter components of the same range group"""
    R, N, ps = pos.shape
    ctx = psg.Context(0)
    ctx.set_layout(R, N, N, ps, 4)
    grp = [("range", first, count)]
    ctx.set_cvs([{"type": psg.CV_RGYR, "groups": grp}] +
                [{"type": psg.CV_COM_COMPONENT, "groups": grp, "axis": a} for a in range(3)], atom_weight=weight)
    xi = torch.empty((R, 4), dtype=torch.float32, device="cuda")
    ctx.cv_eval(torch.from_numpy(pos).cuda(), xi, None)
    ctx.sync_check()
    out = xi.cpu().numpy()
    ctx.close()
    return out


def _definition(pos, first, count, weight):
    """PAPER.md:L188-L189 written out in binary64 (numpy): barycenter and radius of gyration of the range"""
    x = pos[:, first:first + count, :3].astype(np.float64)
    w = np.ones(count) if weight is None else weight[first:first + count].astype(np.float64)
    c = (w[None, :, None] * x).sum(1) / w.sum()
    rg = np.sqrt((w[None, :] * ((x - c[:, None, :]) ** 2).sum(2)).sum(1) / w.sum())
    return rg, c


CASES = [  # (seed, R, N, pos_stride, first, count, weighted): several tiles of 2,048 atoms and a ragged tail
    (11, 5, 40000, 4, 1237, 30011, True),
    (12, 3, 12000, 3, 517, 9000, False),     # fewer replicas, fewer blocks, other stride: stale records of call 1 lie behind
]


def test_static_scratch_entry_point_matches_psg_cv_eval_on_two_calls_in_a_row(torch, psg):
    ref, inputs, outs = [], [], []
    for seed, R, N, ps, first, count, weighted in CASES:
        pos = _positions(seed, R, N, ps)
        weight = np.random.default_rng(seed + 100).uniform(1.0, 16.0, size=N).astype(np.float32) if weighted else None
        ref.append((_existing_path(torch, psg, pos, first, count, weight), _definition(pos, first, count, weight)))
        inputs.append((torch.from_numpy(pos).cuda(), None if weight is None else torch.from_numpy(weight).cuda(), first, count))
        outs.append((torch.full((R,), -1.0, dtype=torch.float32, device="cuda"),
                     torch.full((R, 4), -1.0, dtype=torch.float64, device="cuda")))
    torch.cuda.synchronize()

    def call(k):
        d_pos, d_w, first, count = inputs[k]
        psg.range_rgyr_static(d_pos, first, count, weight=d_w, xi=outs[k][0], center=outs[k][1])

    # two calls in a row on one stream, no synchronisation between them: the second reuses the array the first filled
    call(0)
    call(1)
    torch.cuda.synchronize()
    first_bits = [(o[0].cpu().numpy().copy(), o[1].cpu().numpy().copy()) for o in outs]
    for k, (seed, R, N, ps, first, count, weighted) in enumerate(CASES):
        xi, cen = first_bits[k]
        (xi_ctx, (rg64, c64)) = ref[k]
        assert_close(xi, xi_ctx[:, 0], f"call {k}: Rg vs psg_cv_eval")
        assert_close(cen[:, :3].astype(np.float32), xi_ctx[:, 1:4], f"call {k}: barycenter vs psg_cv_eval")
        assert_close(xi, rg64, f"call {k}: Rg vs the binary64 definition")
        assert_close(cen[:, :3], c64, f"call {k}: barycenter vs the binary64 definition")
        assert np.all(np.abs(xi - xi_ctx[:, 0]) <= np.maximum(REL * np.abs(xi_ctx[:, 0]), ABS))

    # again, in the other order, with the outputs poisoned: the same bits whatever the array held before, and the
    # library took no device memory for it (cudaMalloc would show up in the driver's free-memory figure)
    for o in outs:
        o[0].fill_(-7.0); o[1].fill_(-7.0)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    call(1)
    call(0)
    call(0)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "the no-allocation entry point changed the device's free memory"
    for k in range(len(CASES)):
        assert np.array_equal(outs[k][0].cpu().numpy(), first_bits[k][0]), f"call {k}: Rg depends on the scratch array's old contents"
        assert np.array_equal(outs[k][1].cpu().numpy(), first_bits[k][1]), f"call {k}: barycenter depends on the scratch array's old contents"


def test_static_scratch_entry_point_rejects_sizes_beyond_its_array(torch, psg):
    L = psg.load_library()
    pos = torch.zeros((1, 4096, 4), dtype=torch.float32, device="cuda")
    xi = torch.full((1,), -3.0, dtype=torch.float32, device="cuda")
    vp = ctypes.c_void_p
    # 16,385 replicas x 1 block, and 1 replica x 16,385 blocks: one record more than PSG_STATIC_MAX_BLOCKS (rejected on the
    # host before anything is launched, so the small buffers are never touched)
    for R, stride, count in ((16385, 4096, 2048), (1, 16385 * 2048, 16384 * 2048 + 1)):
        rc = L.psg_range_rgyr_static(0, None, vp(pos.data_ptr()), 4, R, stride, 0, count, None, vp(xi.data_ptr()), None)
        assert rc == -4, rc                                   # PSG_ECAPACITY
        msg = L.psg_static_last_error().decode()
        assert "PSG_STATIC_MAX_BLOCKS" in msg and "16385" in msg, msg
    # exactly the maximum is accepted: 8 replicas x 2,048 blocks = 16,384 records
    big = torch.zeros((8, 2048 * 2048, 3), dtype=torch.float32, device="cuda")
    big[..., 0] = 1.0
    out = torch.empty((8,), dtype=torch.float32, device="cuda")
    psg.range_rgyr_static(big, 0, 2048 * 2048, xi=out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), np.zeros(8, np.float32))   # every atom at (1, 0, 0): Rg = 0 exactly
    for bad in (dict(ps=5), dict(R=0), dict(first=-1), dict(count=0), dict(count=4097)):
        a = dict(ps=4, R=1, first=0, count=4096)
        a.update(bad)
        rc = L.psg_range_rgyr_static(0, None, vp(pos.data_ptr()), a["ps"], a["R"], 4096, a["first"], a["count"], None, vp(xi.data_ptr()), None)
        assert rc == -1, (bad, rc)                            # PSG_EINVAL
    torch.cuda.synchronize()
    assert float(xi.cpu()[0]) == -3.0                         # no rejected call wrote anything
