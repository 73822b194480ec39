"""The entry point that allocates nothing (include/sap_mesh.h, sap_chamfer_nn_static): the exhaustive nearest-neighbour
search of the Chamfer distance (reading M6) with its scratch -- one (distance, index) key per query -- in
the library's file-scope static device array instead of a handle's workspace.  Checked against the existing path,
sap_chamfer in SAP_NN_BRUTE mode through a handle: the indices bit for bit, the distances through the loss
(mean_i d2_a + mean_k d2_b) within the tolerance of tests/test_gpu_mesh.py, on TWO calls in a row with different sets
(the array keeps the keys of the call before: the second result shows that a call resets what it uses).

Collected last on purpose (the suite runs with pytest -x): passes alone in a fresh process and after the other tests."""
import ctypes

import numpy as np
import pytest

from paper_2106_03452_b200 import inputs


def _sets(case):
    """two calls in a row: (a, b) of the first, (a, b) of the second -- the second with FEWER queries and nearer sets, so a
    key left over from the first call would win the atomicMin if it were not reset"""
    if case == "clouds":
        a1, _ = inputs.make_cloud("torus", 20000, seed=11)
        b1, _ = inputs.make_cloud("ellipsoids3", 3000, seed=12)
        a2, _ = inputs.make_cloud("sphere", 7001, seed=13)
        b2, _ = inputs.make_cloud("sphere", 2999, seed=14)
    else:
        rng = np.random.default_rng(5)
        a1 = rng.uniform(0, 1, (37, 3)).astype(np.float32)
        b1 = rng.uniform(0, 1, (4000, 3)).astype(np.float32)
        a2 = rng.uniform(0, 1, (1, 3)).astype(np.float32)
        b2 = rng.uniform(0, 1, (1, 3)).astype(np.float32)
    return (a1, b1), (a2, b2)


@pytest.mark.gpu
@pytest.mark.parametrize("case", ["clouds", "tiny"])
def test_static_scratch_search_matches_the_handle_path_on_two_calls_in_a_row(case):
    import torch
    from paper_2106_03452_b200 import mesh
    from paper_2106_03452_b200.mesh import Mesh
    calls = _sets(case)
    cap = max(max(a.shape[0], b.shape[0]) for a, b in calls)
    h = Mesh(8, 8, 8, cap)
    h.set_search("brute")
    # the existing path first, both calls; then the new entry point, both calls back to back on one stream with outputs
    # allocated BEFORE the first call (nothing is allocated between or inside the two calls)
    want = []
    for a, b in calls:
        ta, tb = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
        loss, _, nn_a, nn_b = h.chamfer(ta, tb, want_grad=False, want_nn=True)
        torch.cuda.synchronize()
        want.append((ta, tb, loss.item(), nn_a.cpu().numpy(), nn_b.cpu().numpy()))
    outs = []
    for ta, tb, *_ in want:
        na, nb = ta.shape[0], tb.shape[0]
        outs.append((torch.full((na,), -7, dtype=torch.int32, device="cuda"), torch.full((na,), -1.0, device="cuda"),
                     torch.full((nb,), -7, dtype=torch.int32, device="cuda"), torch.full((nb,), -1.0, device="cuda")))
    warm = torch.rand((3, 3), device="cuda")      # set-up of the device (the array's address, kernel loading) is not the claim
    mesh.nn_static(warm, warm, torch.empty((3,), dtype=torch.int32, device="cuda"), torch.empty((3,), device="cuda"))
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    for (ta, tb, *_), (nna, d2a, nnb, d2b) in zip(want, outs):
        mesh.nn_static(ta, tb, nna, d2a)     # a -> b
        mesh.nn_static(tb, ta, nnb, d2b)     # b -> a: a second use of the same array inside one Chamfer evaluation
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before and torch.cuda.mem_get_info()[0] >= free_before   # the device lost no memory
    for (ta, tb, loss, nn_a, nn_b), (nna, d2a, nnb, d2b) in zip(want, outs):
        assert np.array_equal(nna.cpu().numpy(), nn_a) and np.array_equal(nnb.cpu().numpy(), nn_b)   # index work: bit-exact
        got = d2a.double().mean().item() + d2b.double().mean().item()
        assert abs(got - loss) <= 1e-5 * loss
        # the distance belongs to the index (float32 arithmetic of the kernel: three products, two fused adds)
        for q, t, nn, d2 in ((ta, tb, nna, d2a), (tb, ta, nnb, d2b)):
            ref = ((q.double() - t[nn.long()].double()) ** 2).sum(1)
            assert torch.all((d2.double() - ref).abs() <= 1e-6 * ref + 1e-12)
    h.close()


@pytest.mark.gpu
def test_static_scratch_search_rejects_what_does_not_fit_and_takes_the_maximum():
    import torch
    from paper_2106_03452_b200 import mesh
    L = mesh.lib()
    big = mesh.NN_STATIC_MAX_QUERIES
    q = torch.rand((big + 1, 3), device="cuda")
    t = torch.rand((64, 3), device="cuda")
    nn = torch.empty((big + 1,), dtype=torch.int32, device="cuda")
    d2 = torch.empty((big + 1,), device="cuda")
    with pytest.raises(mesh.SapError) as e:
        mesh.nn_static(q, t, nn, d2)
    assert e.value.status == 1 and "SAP_NN_STATIC_MAX_QUERIES = 262144" in str(e.value)
    vp = ctypes.c_void_p
    assert L.sap_chamfer_nn_static(None, 1, vp(t.data_ptr()), 64, vp(nn.data_ptr()), vp(d2.data_ptr()), None) == 1
    assert L.sap_chamfer_nn_static(vp(q.data_ptr()), 5, vp(t.data_ptr()), 0, vp(nn.data_ptr()), vp(d2.data_ptr()), None) == 1
    assert L.sap_chamfer_nn_static(vp(q.data_ptr()), -1, vp(t.data_ptr()), 64, vp(nn.data_ptr()), vp(d2.data_ptr()), None) == 1
    # exactly the maximum: every key of the array in use; checked against a plain torch search on a sample of the queries
    qm, nnm, d2m = q[:big], nn[:big], d2[:big]
    mesh.nn_static(qm, t, nnm, d2m)
    torch.cuda.synchronize()
    idx = torch.cat([torch.arange(0, 300, device="cuda"), torch.arange(big - 300, big, device="cuda")])
    dist = ((qm[idx, None, :].double() - t[None, :, :].double()) ** 2).sum(2)
    ref_d, ref_i = dist.min(1)
    got_d = ((qm[idx].double() - t[nnm[idx].long()].double()) ** 2).sum(1)
    assert torch.all((got_d - ref_d).abs() <= 1e-6 * ref_d + 1e-12)       # the same neighbour up to float32 near-ties
    assert (nnm[idx].long() != ref_i).double().mean().item() <= 1e-2
    assert int(nnm.min()) >= 0 and int(nnm.max()) < 64


def test_static_scratch_entry_point_validates_before_cuda():
    """no GPU needed: the argument checks come before the first CUDA call"""
    from paper_2106_03452_b200 import build, mesh
    build.build()
    L = mesh.lib()
    one = ctypes.c_void_p(8)    # never dereferenced: every call below is rejected on its sizes
    assert L.sap_chamfer_nn_static(None, 1, None, 1, None, None, None) == 1
    assert L.sap_chamfer_nn_static(one, mesh.NN_STATIC_MAX_QUERIES + 1, one, 1, one, one, None) == 1
    assert b"SAP_NN_STATIC_MAX_QUERIES" in L.sap_mesh_last_error(None)
    assert L.sap_chamfer_nn_static(one, 0, one, 1, one, one, None) == 0      # an empty query set enqueues nothing
    assert L.sap_chamfer_nn_static(one, 3, one, 0, one, one, None) == 1
