"""-m gpu: behaviour at the boundary that the per-config parity tests do not reach.

  * open / inward-wound meshes: the DEGENERATE branch of step 9 (fate -3) on the GPU, ray for ray the oracle's;
  * MCX_ERR_CAPACITY: a ray through the apex of a fan of more triangles than the per-ray end-point scratch holds is
    dropped, counted, and reported by the calls include/mcx.h names, until mcx_tally_reset;
  * the absorber gate's first launch on a fresh handle (the block that finishes its first tile first chooses the gate
    for all) with a foreign kernel co-running on another stream: exact ray counts every time;
  * two handles tracing disjoint ray-index windows sum to one handle tracing the whole range (the multi-GPU gather/add
    of PAPER.md:77, 110 on device buffers).
"""
import numpy as np
import pytest

from _parity import assert_tally_parity
from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu

H = (1 / 64, 3 / 128, 1 / 128)


def _flat(mu):
    return {"E": np.array([1.0, 1000.0]), "mu": np.array([mu, mu])}


def mesh_instrument(W, solid, n_rays, target=0.2):
    src = W.source("point", "target", "mono", target_w=target, target_h=target, target_dist=1.0, E0=30.0)
    det = W.detector(-0.1, 0.1, -0.1, 0.1, 16, 16, 0.0, 60.0, 1, T=(0, 0, 1.0))
    return W.instrument("mesh_edge_case", [src, W.solids([solid]), det], [None, _flat(80.0)], n_rays)


def test_open_and_inward_meshes_give_the_oracles_degenerate_rays(M, O, W):
    V, F = W.cube_mesh(*H)
    top = np.array([all(V[v][2] > 0 for v in f) for f in F])
    for tris in (F[~top], F[:, [0, 2, 1]]):
        inst = mesh_instrument(W, W.solid_mesh(V, tris, 1, 0, T=(0, 0, 0.5)), 30_000)
        o = O.trace(inst, dump=True)
        assert 1000 < o["degenerate"] < 29_000                  # the branch is really taken, and not by every ray
        st = check(M, O, W, inst, 30_000)                       # fates (incl. -3), bins, weights, counters: all equal
        assert st["n_diff"] == 0
    # rotated open mesh, both lane schedules, larger mesh with one triangle removed
    rng = np.random.default_rng(5)
    Vb, Fb = W.bumpy_sphere(rng, 3, 20e-3)
    inst = mesh_instrument(W, W.solid_mesh(Vb, Fb[5:], 1, 0, R=W.random_rotation(rng), T=(0, 0, 0.5)), 60_000, target=0.1)
    o = O.trace(inst, dump=True)
    assert o["degenerate"] > 0
    check(M, O, W, inst, 60_000)


def fan_cone(W, k, r=5e-3, h=4e-3):
    """Closed cone: apex (0, 0, -h), a ring of k vertices at z = 0, base centre (0, 0, 0).  2k triangles, k of them
    around the apex and k around the base centre."""
    ang = 2 * np.pi * np.arange(k) / k
    V = np.vstack([[0.0, 0.0, -h], [0.0, 0.0, 0.0], np.stack([r * np.cos(ang), r * np.sin(ang), np.zeros(k)], axis=1)])
    F = []
    for i in range(k):
        a, b = 2 + i, 2 + (i + 1) % k
        F += [(0, b, a), (1, a, b)]
    F = np.array(F, dtype=np.int32)
    n = np.cross(V[F[:, 1]] - V[F[:, 0]], V[F[:, 2]] - V[F[:, 0]])
    ctr = (V[F[:, 0]] + V[F[:, 1]] + V[F[:, 2]]) / 3.0 - np.array([0, 0, -h / 3])
    flip = np.einsum("ij,ij->i", n, ctr) < 0
    F[flip] = F[flip][:, [0, 2, 1]]
    return V, F


def test_capacity_overflow_is_reported(M, O, W):
    import torch
    V, F = fan_cone(W, 64)
    cone = W.solid_mesh(V, F, 1, 0, T=(0, 0, 0.5))
    # target of zero size: every ray runs down the axis, through the apex (64 triangles) and the base centre (64 more)
    inst = mesh_instrument(W, cone, 3000, target=0.0)
    o = O.trace(inst, n=50, dump=True)
    assert o["detected"] == 50 and abs(o["dump"]["p"][0] - np.exp(-80.0 * 4e-3)) < 1e-13     # the oracle has no capacity
    g = M.Instrument(inst)
    g.status()
    g.trace(3000)
    torch.cuda.synchronize()
    for call in (lambda: g.tally(0), lambda: g.counters(), lambda: g.status(), lambda: g.trace(10)):
        with pytest.raises(M.McxError) as e:
            call()
        assert e.value.status == M.binding.MCX_ERR_CAPACITY
    with pytest.raises(M.McxError) as e:
        g.status()
    assert "3010 rays" in str(e.value)
    c = g.counters(allow_capacity=True)
    assert c["overflows"] == 3010 and c["degenerate"] == 3010 and c["detected"] == 0
    assert np.all(g.trace_dump(0, 100)["fate"] == M.binding.FATE_DEGENERATE)
    g.reset()                                                   # forgets it
    g.status()
    assert int(g.tally(0)[0].sum()) == 0
    g.close()
    # the same cone seen off-axis never overflows and matches the oracle
    check(M, O, W, mesh_instrument(W, cone, 40_000, target=0.04), 40_000)
    # 24 triangles around each apex (48 raw hits) just fit the largest scratch of a 1-mesh group? No: the scratch of
    # one mesh is 16 end points; 6 + 6 fits
    V6, F6 = fan_cone(W, 6)
    check(M, O, W, mesh_instrument(W, W.solid_mesh(V6, F6, 1, 0, T=(0, 0, 0.5)), 2000, target=0.0), 2000)


def test_gate_choice_on_first_launch_with_a_corunning_kernel(M, O, W):
    import torch
    inst = W.config0()
    side = torch.cuda.Stream()
    a = torch.randn(2048, 2048, device="cuda")
    expect = {}
    for rep in range(40):
        n = (3000, 20_000, 70_001, 300_000)[rep % 4]
        if n not in expect:
            o = O.trace(inst, n=n)
            expect[n] = (o["N"][0].copy(), o["absorbed"].copy(), o["detected"])
        g = M.Instrument(inst)                                  # fresh handle: the gate is not known yet
        with torch.cuda.stream(side):
            for _ in range(4):
                a = (a @ a).clamp_(-1, 1)                       # foreign work: blocks of the trace start staggered
        g.trace(n)
        N = g.tally(0)[0].cpu().numpy().view(np.uint64)
        c = g.counters()
        assert np.array_equal(N, expect[n][0]), f"rep {rep}: counts differ"
        assert np.array_equal(c["absorbed"].astype(np.uint64), expect[n][1]) and c["detected"] == expect[n][2]
        g.trace(n, first=n)                                     # second launch: starts with the remembered gate
        assert g.counters()["detected"] + int(g.counters()["absorbed"].sum()) == 2 * n
        g.close()
    torch.cuda.synchronize()


def test_two_handles_over_disjoint_windows_sum_to_the_whole(M, O, W):
    """The paper's scatter-gather (PAPER.md:77 "all results are added", :110 multi-GPU through the same split): rank r
    traces its share of the ray-index range on its own replica, then the (N, p, p2) arrays are summed.  Here both
    replicas live on the one GPU there is; the sum runs on device tensors, as the NCCL reduce of bench.py does."""
    from paper_2410_08747_b200.shard import ray_range
    for k, n in ((1, 300_000), (4, 60_000)):
        inst = W.config(k, small=True)
        whole = M.Instrument(inst)
        whole.trace(n)
        ref = [t.clone() for t in whole.tally(0)]
        whole.close()
        parts = []
        for r in range(2):
            first, count = ray_range(r, 2, n, "strong")
            h = M.Instrument(inst)
            h.trace(count, first=first)
            parts.append([t.clone() for t in h.tally(0)])
            h.close()
        tot = [a + b for a, b in zip(*parts)]
        assert bool((tot[0] == ref[0]).all())                   # integer counts exact
        W_tot, W2_tot = float(ref[1].sum()), float(ref[2].sum())
        assert float((tot[1] - ref[1]).abs().max()) <= 1e-9 * W_tot
        assert float((tot[2] - ref[2]).abs().max()) <= 1e-9 * W2_tot
        o = O.trace(inst, n=n)
        assert_tally_parity((tot[0].cpu().numpy().view(np.uint64), tot[1].cpu().numpy(), tot[2].cpu().numpy()),
                            (o["N"][0], o["P"][0], o["P2"][0]), exact_N=False)
