"""tbsma_kinetic_tensor_noalloc (include/tbsma.h): the one entry point of the library that allocates no device memory.

It exists for callers that cannot call cudaMalloc: code plugged into an MD engine or framework whose own pool already
holds the GPU's memory, analysis hooks inside a loop that must not take cudaMalloc's device-wide synchronisation, jobs
with a fixed memory budget.  Its working memory is a fixed 784 KiB array inside the library's device code, one per GPU,
shared by every call and never cleared between calls, so what has to be shown is that (a) it computes what the
context-based tbsma_kinetic_tensor computes and (b) a call is not disturbed by what the call before it left in that array
-- hence several calls in a row on batches of different shapes, each compared with the existing path at the tolerance
tests/test_gpu_parity.py uses for the kinetic tensor (rtol 1e-11, atol 1e-12: both sum the same fp64 products, only the
order of the additions differs).

This file is named so that pytest collects it last: the GPU suite runs with -x, and a failure here must not hide the parity
tests.  It passes on its own in a fresh process (the first call then also performs the per-GPU set-up, the look-up of the
array's device address) and after the other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1311_3890_b200 import workloads as W

torch = pytest.importorskip("torch")

RTOL, ATOL = 1e-11, 1e-12      # test_stress_and_kinetic_tensor_match_oracle's bar


def test_sizes_beyond_the_fixed_scratch_are_rejected():
    """no GPU needed: the size check comes before any CUDA call, names its own error code, and explains itself"""
    from paper_1311_3890_b200 import binding as B
    L = B.lib()
    big = B.NOALLOC_MAX_REPLICAS + 1
    one = C.c_void_p(256)                      # never dereferenced: the call returns before touching the GPU
    assert L.tbsma_kinetic_tensor_noalloc(one, one, one, 10 * big, big, 196.97, one, None) == B.ELIMIT
    assert L.tbsma_kinetic_tensor_noalloc(one, one, one, 2 ** 31, 4, 196.97, one, None) == B.ELIMIT
    assert "fixed capacity" in B.strerror(B.ELIMIT)
    assert L.tbsma_kinetic_tensor_noalloc(one, one, one, -1, 4, 196.97, one, None) == B.EINVAL
    assert L.tbsma_kinetic_tensor_noalloc(one, one, one, 100, 4, 0.0, one, None) == B.EINVAL
    assert L.tbsma_kinetic_tensor_noalloc(one, one, None, 100, 4, 196.97, one, None) == B.EINVAL
    assert L.tbsma_kinetic_tensor_noalloc(None, None, None, 0, 0, 196.97, None, None) == B.OK     # empty batch


@pytest.mark.gpu
def test_no_alloc_kinetic_tensor_matches_the_context_path_on_calls_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1311_3890_b200 import binding as B

    def batch(w):
        """device tensors of a workload and the kinetic tensor by the existing, context-based path"""
        st = B.DeviceState(w)
        ctx = B.make_context(w)
        ref = torch.full((w.n_replicas, 6), -1.0, dtype=torch.float64, device="cuda")
        ctx.kinetic_tensor(st.pos, st.vel, ref)
        torch.cuda.synchronize()
        off = torch.from_numpy(np.ascontiguousarray(w.offsets, dtype=np.int32)).cuda()
        return st, off, ref.cpu().numpy()

    # three shapes, so that consecutive calls use different numbers of replicas and of slices per replica and find
    # each other's tickets and partial sums in the array: 4 long wires with grips at 10 K / 298 K (11 slices each), a
    # ragged batch of 37 short hot wires (3 slices), one wire alone
    wa, wb, wc = W.config3(4, seed=23), W.config4(37, seed=31), W.config2()
    (sa, oa, ra), (sb, ob, rb), (sc, oc, rc) = batch(wa), batch(wb), batch(wc)
    assert np.all(ra[:, :3] > 0) and np.all(rb[:, :3] > 0) and np.all(rc[:, :3] > 0)
    outs = []
    for st, off, R in ((sa, oa, 4), (sb, ob, 37), (sa, oa, 4), (sc, oc, 1), (sb, ob, 37)):
        k = torch.full((R, 6), float("nan"), dtype=torch.float64, device="cuda")     # the call must overwrite every entry
        B.kinetic_tensor_noalloc(st.pos, st.vel, off, k)                             # same stream: calls do not overlap
        outs.append(k)
    torch.cuda.synchronize()
    outs = [k.cpu().numpy() for k in outs]
    for got, ref in zip(outs, (ra, rb, ra, rc, rb)):
        assert np.all(np.isfinite(got))
        assert np.allclose(got, ref, rtol=RTOL, atol=ATOL)
    # the sums are added in a fixed order: the same batch gives the same bits whatever ran in between
    assert np.array_equal(outs[0], outs[2]) and np.array_equal(outs[1], outs[4])

    # an empty replica in the middle of a batch gets zeros; a replica of grip atoms only as well
    off = torch.tensor([0, 700, 700, 1500], dtype=torch.int32, device="cuda")
    pos = sc.pos[:1500].clone()
    pos.view(torch.int32)[700:, 3] = 1                                               # flag 1: fixed grip
    k = torch.full((3, 6), float("nan"), dtype=torch.float64, device="cuda")
    B.kinetic_tensor_noalloc(pos, sc.vel[:1500].contiguous(), off, k)
    torch.cuda.synchronize()
    k = k.cpu().numpy()
    assert np.all(k[0, :3] > 0) and np.all(k[1:] == 0.0)

    # beyond the fixed capacity: a clear error through the binding, nothing launched
    with pytest.raises(B.TbsmaError) as e:
        R = B.NOALLOC_MAX_REPLICAS + 1
        B.kinetic_tensor_noalloc(sc.pos, sc.vel, torch.zeros(R + 1, dtype=torch.int32, device="cuda"),
                                 torch.zeros(R, 6, dtype=torch.float64, device="cuda"))
    assert e.value.code == B.ELIMIT and "fixed capacity" in str(e.value)
