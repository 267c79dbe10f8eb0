"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the fp64 oracle on
the same seeded inputs.  Bars (BASELINE.json north_star): neighbour sets bit-exact; per-atom
force |dF| <= 1e-4 eV/A + 1e-5 |F|; total energy relative error <= 1e-6; trajectories within
1e-3 A RMS after 100 steps.  Everything is compared in tag (original index) space."""
import math

import numpy as np
import pytest

import oracle
from paper_1311_3890_b200 import workloads as W

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

KB, ACC, MASS = 8.617333262e-5, 9.648533212e-3, 196.96657
F_ABS, F_REL, E_REL, TRAJ_RMS = 1e-4, 1e-5, 1e-6, 1e-3


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1311_3890_b200 import binding
    return binding


VARIANTS = [1, 2]     # 1 = global-gather lists, 2 = shared-memory tiles (layer tiles of thin wires, box tiles otherwise)


def setup(B, w, max_nb=96, variant=0, tile=None, stagger=True, box=False):
    if variant == 2 and np.any(w.periodic) and float((w.box_hi - w.box_lo)[w.periodic != 0].min()) < 3 * 9.81:
        pytest.skip("the shared-memory tile variant needs three cells of r_cut + skin + S along a periodic axis")
    ctx = B.make_context(w, max_nb)
    ctx.set_variant(variant)
    if tile:
        ctx.set_tile(*tile)
    if box:
        ctx.set_tile_box(True)
    ctx.set_stagger(stagger)
    st = B.DeviceState(w)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    if variant:
        assert ctx.get_variant() == variant
    return ctx, st


def gpu_neighbors(B, ctx, st):
    counts = torch.zeros(ctx.n, dtype=torch.int32, device="cuda")
    lst = torch.full((ctx.n, ctx.max_neighbors), -1, dtype=torch.int32, device="cuda")
    ctx.get_neighbors(st.tag, counts, lst)
    torch.cuda.synchronize()
    return counts.cpu().numpy(), lst.cpu().numpy()


def assert_same_sets(cg, lg, co, lo):
    assert np.array_equal(cg, co)
    for i in range(len(cg)):
        assert np.array_equal(np.sort(lg[i, :cg[i]]), lo[i, :co[i]]), i


def assert_forces(fg, fo):
    err = np.linalg.norm(fg - fo, axis=1)
    tol = F_ABS + F_REL * np.linalg.norm(fo, axis=1)
    assert np.all(err <= tol), f"max force error {err.max():.3e}"
    return err.max()


def small_bulk(ncell=6, seed=5, a=4.08):
    """periodic block, positions wrapped in fp32 like config 5a"""
    w = W.config5a(ncell, seed)
    return w


WORKLOADS = {
    "config1": lambda: W.config1(),
    "config2": lambda: W.config2(),
    "config4_ragged": lambda: W.config4(5, seed=9),
    "config3_small": lambda: W.config3(2, seed=3, length=60.0),
    "bulk_6": lambda: small_bulk(6),
    "bulk_4_two_cells": lambda: small_bulk(4),       # 16.32 A box: only 2 cells per axis
    "bulk_9": lambda: small_bulk(9),
    "bulk_13": lambda: small_bulk(13),               # 53 A box: five cells of the tile variant per axis, boxes of 1 cell
    "bulk_18": lambda: small_bulk(18),               # 73 A box: seven cells, boxes of 2 x 2 x 2 cells
    "thick_wire": lambda: W.config5b(length=80.0),   # 6 nm wire: layers do not fit a tile image, boxes of cells
}


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("name", list(WORKLOADS))
def test_neighbor_sets_bit_exact(B, name, variant):
    w = WORKLOADS[name]()
    ctx, st = setup(B, w, variant=variant)
    cg, lg = gpu_neighbors(B, ctx, st)
    co, lo = oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert ctx.status() & B.FLAG_NLIST_OVERFLOW == 0
    assert_same_sets(cg, lg, co, lo)
    # tags are a permutation that keeps every atom inside its replica
    tag = st.tag.cpu().numpy()
    assert np.array_equal(np.sort(tag), np.arange(w.n_atoms))
    for r in range(w.n_replicas):
        s = slice(w.offsets[r], w.offsets[r + 1])
        assert tag[s].min() >= w.offsets[r] and tag[s].max() < w.offsets[r + 1]
    entries, pairs = ctx.count_pairs(st.pos)
    assert entries == co.sum()
    cc, _ = oracle.neighbors(w.pos4, w.r_cut, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert pairs == cc.sum()


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("name", list(WORKLOADS))
def test_force_energy_virial_parity(B, name, variant):
    w = WORKLOADS[name]()
    ctx, st = setup(B, w, variant=variant)
    ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    o = oracle.compute(w.x64(), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, periodic=w.periodic)
    fe = st.untag(st.force)
    assert_forces(fe[:, :3].astype(np.float64), o["f"])
    assert np.abs(fe[:, 3] - o["e_atom"]).max() <= 2e-6 * np.abs(o["e_atom"]).max() + 1e-6
    e = st.e_rep.cpu().numpy()
    assert np.all(np.abs(e - o["e_rep"]) <= E_REL * np.abs(o["e_rep"]))
    wv = st.w_rep.cpu().numpy()
    scale = np.abs(o["w_rep"][:, :3]).sum(1, keepdims=True) + w.n_atoms / w.n_replicas * 1e-3
    assert np.all(np.abs(wv - o["w_rep"]) <= 2e-5 * scale)
    # positions were only permuted (and wrapped), never changed, by the build
    assert np.array_equal(st.untag(st.pos)[:, :3], w.pos4[:, :3])
    # energy-only call (virial = NULL) gives the same forces bit for bit
    f2 = torch.zeros_like(st.force)
    ctx.compute(st.pos, f2, st.e_rep, None)
    torch.cuda.synchronize()
    assert torch.equal(f2, st.force)


@pytest.mark.parametrize("variant", VARIANTS)
def test_paper_cutoff_5p8(B, variant):
    """the paper's own r_cut = 5.8 A, r_buff = 0.29 A"""
    w = W.config1()
    w.r_cut, w.skin = 5.8, 0.29
    ctx, st = setup(B, w, variant=variant)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    o = oracle.compute(w.x64(), 5.8)
    assert_forces(st.untag(st.force)[:, :3].astype(np.float64), o["f"])
    assert abs(st.e_rep.item() - o["e_rep"][0]) <= E_REL * abs(o["e_rep"][0])
    cg, lg = gpu_neighbors(B, ctx, st)
    co, lo = oracle.neighbors(w.pos4, 5.8 + 0.29)
    assert_same_sets(cg, lg, co, lo)


@pytest.mark.parametrize("variant", VARIANTS)
def test_degenerate_systems(B, variant):
    # single atom, dimer inside / outside the cutoff, an empty replica in the middle (reading A5)
    x = np.array([[0, 0, 0], [10, 0, 0], [12.5, 0, 0], [30, 0, 0], [38, 0, 0]], dtype=np.float64)
    offs = np.array([0, 1, 3, 3, 5], dtype=np.int32)
    lo = np.array([[-5, -5, -5], [5, -5, -5], [0, 0, 0], [25, -5, -5]], np.float32)
    hi = np.array([[5, 5, 5], [20, 5, 5], [1, 1, 1], [45, 5, 5]], np.float32)
    w = W.Workload("degenerate", W.pack_pos4(x), W.pack_vel4(np.zeros((5, 3)), W.pack_pos4(x)), offs, lo, hi,
                   np.zeros((4, 3), np.uint8), np.zeros(4, np.float32), np.arange(4, dtype=np.uint64), np.zeros(4))
    ctx, st = setup(B, w, variant=variant)
    ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
    torch.cuda.synchronize()
    o = oracle.compute(x, 7.0, offsets=offs, lo=lo, hi=hi, periodic=0)
    fe = st.untag(st.force)
    assert np.all(fe[[0, 3, 4]] == 0) and np.all(np.isfinite(fe))
    assert_forces(fe[:, :3].astype(np.float64), o["f"])
    assert np.allclose(st.e_rep.cpu().numpy(), o["e_rep"], rtol=1e-6, atol=0)
    assert st.e_rep[0].item() == 0 and st.e_rep[2].item() == 0 and st.e_rep[3].item() == 0
    assert ctx.status() == 0


@pytest.mark.parametrize("variant", VARIANTS)
def test_list_overflow_is_flagged(B, variant):
    w = W.config1()
    ctx = B.make_context(w, 32)            # far too small for r = 7.3 A (up to 86 partners)
    ctx.set_variant(variant)
    st = B.DeviceState(w)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    assert ctx.status() & B.FLAG_NLIST_OVERFLOW
    seen = ctx.get_stats()["max_neighbors_seen"]
    # the tile variant filters its list from a candidate list that overflowed first (capacity scales with max_neighbors)
    assert seen == 86 if variant == 1 else 32 < seen <= 86
    ctx.clear_status()
    assert ctx.status() == 0


def test_call_order_and_arguments(B):
    w = W.config1()
    ctx = B.make_context(w)
    st = B.DeviceState(w)
    with pytest.raises(B.TbsmaError) as e:
        ctx.compute(st.pos, st.force)
    assert e.value.code == B.ESTATE
    with pytest.raises(B.TbsmaError) as e:
        ctx.build_neighbors(st.pos, st.vel, st.tag)
    assert e.value.code == B.ESTATE
    bad = B.Context()
    with pytest.raises(B.TbsmaError) as e:        # periodic box shorter than 2 (r_cut + skin)
        bad.set_system([0, 10], 0.0, 14.0, 1)
    assert e.value.code == B.EINVAL


def run_gpu_md(B, w, n_steps, use_run=True, graph=True, virial=False, variant=0, tile=None, overlap=2,
               stagger=True, async_inner=True, conditional=True, max_nb=96):
    ctx, st = setup(B, w, max_nb=max_nb, variant=variant, tile=tile, stagger=stagger)
    ctx.set_graph(graph, conditional=conditional)
    ctx.set_overlap(overlap)
    ctx.set_async(async_inner)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        if use_run:
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None,
                       st.slab_rate, w.rebuild_every, st.e_rep, st.w_rep if virial else None, st.ekin)
        else:
            for s in range(n_steps):
                disp = torch.from_numpy(w.slab_rate * (s + 1)).cuda()
                ctx.md_step(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, s, disp, st.e_rep,
                            st.w_rep if virial else None, st.ekin)
    torch.cuda.synchronize()
    return ctx, st


def run_oracle_md(w, n_steps, cells=True, fp32_pred=False):
    md = oracle.MD(w.x64(), w.v64(), w.flags, w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi,
                   periodic=w.periodic, fp32_pred=fp32_pred, cells=cells, zref=w.vel4[:, 3].astype(np.float64))
    for s in range(n_steps):
        md.step(w.dt, w.T.astype(np.float64), w.gamma, w.seed, s, slab_disp=w.slab_rate * (s + 1))
    return md


def traj_rms(xg, xo, box_len=None):
    d = xg - xo
    if box_len is not None:
        d -= np.round(d / box_len) * box_len
    return math.sqrt((d ** 2).sum(1).mean())


@pytest.mark.parametrize("variant", VARIANTS)
def test_trajectory_config1_nve_100_steps(B, variant):
    w = W.config1()
    ctx, st = run_gpu_md(B, w, 100, variant=variant)
    md = run_oracle_md(w, 100)
    assert traj_rms(st.untag(st.pos)[:, :3].astype(np.float64), md.x) <= TRAJ_RMS
    assert abs(st.e_rep.item() - md.e_rep[0]) <= 5e-6 * abs(md.e_rep[0])
    assert abs(st.ekin.item() - md.ekin_rep[0]) <= 1e-3 * md.ekin_rep[0]
    # the forces left in the buffer are those of the final positions
    assert_forces(st.untag(st.force)[:, :3].astype(np.float64),
                  oracle.compute(st.untag(st.pos)[:, :3].astype(np.float64), 7.0)["f"])
    assert ctx.status() == 0
    assert ctx.get_stats()["n_steps"] == 100


@pytest.mark.parametrize("variant", VARIANTS)
def test_trajectory_config2_langevin_grips_pull(B, variant):
    w = W.config2()
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps, variant=variant)
    md = run_oracle_md(w, n_steps)
    xg = st.untag(st.pos)[:, :3].astype(np.float64)
    assert traj_rms(xg, md.x) <= TRAJ_RMS
    vg = st.untag(st.vel)[:, :3].astype(np.float64)
    assert np.abs(vg - md.v).max() < 2e-5
    fl = w.flags
    # grips: fixed atoms never move, pulled atoms sit at zref + D to 1 ulp (H5), v = 0
    assert np.array_equal(xg[fl == 1], w.x64()[fl == 1])
    zt = (w.vel4[fl == 2, 3].astype(np.float64) + w.slab_rate[0] * n_steps).astype(np.float32)
    assert np.array_equal(st.untag(st.pos)[fl == 2, 2], zt)
    assert np.all(vg[fl != 0] == 0)
    stats = ctx.get_stats()
    assert stats["n_replica_builds"] >= 1          # 298 K: atoms pass skin/2 within 100 steps
    assert abs(st.ekin.item() - md.ekin_rep[0]) <= 2e-3 * md.ekin_rep[0]
    assert ctx.status() == 0


@pytest.mark.parametrize("variant", VARIANTS)
def test_md_step_equals_md_run_and_graph_bitwise(B, variant):
    w = W.config2(length=60.0)
    _, a = run_gpu_md(B, w, 40, use_run=True, graph=True, variant=variant)
    _, b = run_gpu_md(B, w, 40, use_run=True, graph=False, variant=variant)
    _, c = run_gpu_md(B, w, 40, use_run=False, variant=variant)
    for s in (b, c):
        assert np.array_equal(a.untag(a.pos), s.untag(s.pos))
        assert np.array_equal(a.untag(a.vel), s.untag(s.vel))
        assert np.array_equal(a.untag(a.force), s.untag(s.force))


@pytest.mark.parametrize("variant", VARIANTS)
def test_replicas_are_independent_and_ragged_batch_matches_single_runs(B, variant):
    # staggering (tbsma_set_stagger) makes a replica's FIRST rebuild depend on its index in the batch, which changes the
    # fp32 summation order, not the physics: switched off here because this test compares bits
    w = W.config4(4, seed=21)
    n_steps = 60
    _, st = run_gpu_md(B, w, n_steps, variant=variant, stagger=False)
    xb = st.untag(st.pos)
    assert len(set(np.diff(w.offsets))) > 1        # really ragged
    for r in range(w.n_replicas):
        single = w.take(r, r + 1)
        _, ss = run_gpu_md(B, single, n_steps, variant=variant, stagger=False)
        s = slice(w.offsets[r], w.offsets[r + 1])
        assert np.array_equal(xb[s], ss.untag(ss.pos))          # bit-identical: no cross-replica effect


@pytest.mark.parametrize("overlap", [1, 2])
@pytest.mark.parametrize("graph", [True, False])
def test_overlapped_list_renewal_is_bitwise_identical(B, graph, overlap):
    """the filter pass beside the gather passes (tbsma_set_overlap: 1 = second stream, 2 = the density pass launched as
    its programmatic dependent) changes nothing: a batch with 10 K and 298 K replicas (so that some rebuild while
    others do not) gives the same bits as the same kernels one after the other"""
    w = W.config3(6, seed=11, length=60.0)
    n_steps = 80
    ca, a = run_gpu_md(B, w, n_steps, variant=2, graph=graph, overlap=overlap, virial=True)
    cb, b = run_gpu_md(B, w, n_steps, variant=2, graph=graph, overlap=0, virial=True)
    sa, sb = ca.get_stats(), cb.get_stats()
    assert sa == sb
    assert 0 < sa["n_replica_builds"] < w.n_replicas * n_steps and sa["n_build_passes"] < n_steps
    for name in ("pos", "vel", "force"):
        assert np.array_equal(a.untag(getattr(a, name)), b.untag(getattr(b, name))), name
    # per-replica sums are added in a fixed order (chunk tree, chunks of a CTA in order, CTAs of a replica in tile order)
    assert np.array_equal(a.e_rep.cpu().numpy(), b.e_rep.cpu().numpy())
    assert np.array_equal(a.ekin.cpu().numpy(), b.ekin.cpu().numpy())
    assert np.array_equal(a.w_rep.cpu().numpy(), b.w_rep.cpu().numpy())
    assert ca.status() == 0 and cb.status() == 0
    md = run_oracle_md(w, n_steps)
    assert traj_rms(a.untag(a.pos)[:, :3].astype(np.float64), md.x) <= TRAJ_RMS


def test_per_replica_sums_are_bitwise_repeatable_and_tile_split_changes_only_their_order(B):
    """a6 in the tile variant: the same run twice gives the same bits in E, E_kin and W of every replica (no atomics);
    several CTAs per tile (tbsma_set_tile_split, what small batches get automatically) leave positions, velocities and
    forces bit-identical and change the per-replica sums only by their fp64 summation order"""
    w = W.config3(3, seed=17, length=60.0)
    n_steps = 40

    def run(split):
        ctx, st = setup(B, w, variant=2)
        if split is not None:
            ctx.set_tile_split(split)
            ctx.build_cells(st.pos, st.vel, st.tag)
            ctx.build_neighbors(st.pos, st.vel, st.tag)
        ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
        torch.cuda.synchronize()
        e0, w0 = st.e_rep.cpu().numpy().copy(), st.w_rep.cpu().numpy().copy()
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate, 0,
                       st.e_rep, st.w_rep, st.ekin)
        torch.cuda.synchronize()
        assert ctx.status() == 0
        return dict(e0=e0, w0=w0, pos=st.untag(st.pos), vel=st.untag(st.vel), force=st.untag(st.force),
                    e=st.e_rep.cpu().numpy().copy(), k=st.ekin.cpu().numpy().copy(), w=st.w_rep.cpu().numpy().copy())

    a, b = run(None), run(None)
    for key in a:
        assert np.array_equal(a[key], b[key]), key
    o = oracle.compute(w.x64(), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi)
    assert np.all(np.abs(a["e0"] - o["e_rep"]) <= E_REL * np.abs(o["e_rep"]))
    assert np.abs(a["w0"] - o["w_rep"]).max() <= 2e-5 * np.abs(o["w_rep"][:, :3]).sum(1).max()
    for split in (1, 3, 7):
        c = run(split)
        for key in ("pos", "vel", "force"):
            assert np.array_equal(a[key], c[key]), (split, key)
        for key in ("e0", "w0", "e", "k", "w"):
            assert np.allclose(a[key], c[key], rtol=1e-12, atol=1e-10), (split, key)


def test_switching_to_the_global_variant_after_a_tile_run(B):
    """after a run in the tile variant some replicas use the second half of the list buffers; rebuilding for the global
    variant (which only has the first) on the same context must not leave them pointing there: no spurious rebuilds,
    no SKIN_VIOLATED, same trajectory as a fresh global-variant context"""
    w = W.config3(4, seed=19, length=60.0)
    ctx, st = run_gpu_md(B, w, 60, variant=2)
    assert ctx.get_variant() == 2 and ctx.get_stats()["n_replica_builds"] > w.n_replicas
    ctx.set_variant(1)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    torch.cuda.synchronize()
    assert ctx.get_variant() == 1
    x0, v0 = st.untag(st.pos), st.untag(st.vel)
    b0 = ctx.get_stats()["n_replica_builds"]
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 60, 5, None, None, 0, st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    assert ctx.get_stats()["n_replica_builds"] - b0 <= w.n_replicas      # not "every replica every step"
    # reference: a fresh context in the global variant from the same state
    w2 = W.Workload(w.name, x0.copy(), v0.copy(), w.offsets, w.box_lo, w.box_hi, w.periodic, w.T, w.seed, np.zeros_like(w.slab_rate),
                    w.gamma, w.dt, w.r_cut, w.skin, 0, {})
    ctx2, st2 = setup(B, w2, variant=1)
    ctx2.compute(st2.pos, st2.force, st2.e_rep, None)
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        ctx2.md_run(st2.pos, st2.vel, st2.force, st2.tag, w.dt, st2.T, w.gamma, st2.seed, 60, 5, None, None, 0, st2.e_rep, None, st2.ekin)
    torch.cuda.synchronize()
    assert np.array_equal(st.untag(st.pos)[:, :3], st2.untag(st2.pos)[:, :3])


def test_fixed_cadence_with_several_replicas_and_chained_runs(B):
    """rebuild_every > 0 on a batch: the staggered first rebuild (for displacement-triggered lists) must not fire and be
    reported as a violated skin; and md_run called in pieces (step0 = 0, 7, 14, ...: one captured graph serves them
    all, the step number of the run lives on the device) gives the bits of one long call"""
    w = W.config3(4, seed=23, length=60.0)
    w.rebuild_every = 10
    n = 42
    ca, a = run_gpu_md(B, w, n, variant=0)
    assert ca.status() == 0
    assert ca.get_stats()["n_build_passes"] == 1 + 5          # the explicit build + steps 0, 10, 20, 30, 40
    ctx, st = setup(B, w)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    torch.cuda.synchronize()
    stream = torch.cuda.Stream()
    rate = st.slab_rate
    with torch.cuda.stream(stream):
        for s0 in range(0, n, 7):
            m = min(7, n - s0)
            disp0 = rate * float(s0)
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, s0, m, disp0, rate, w.rebuild_every,
                       st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    assert np.array_equal(a.untag(a.pos), st.untag(st.pos))
    # and with pieces long enough to go through the captured graph
    ctx3, st3 = setup(B, w)
    ctx3.compute(st3.pos, st3.force, st3.e_rep, None)
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        for s0 in range(0, 40, 10):
            ctx3.md_run(st3.pos, st3.vel, st3.force, st3.tag, w.dt, st3.T, w.gamma, st3.seed, s0, 10, st3.slab_rate * float(s0),
                        st3.slab_rate, w.rebuild_every, st3.e_rep, None, st3.ekin)
        ctx3.md_run(st3.pos, st3.vel, st3.force, st3.tag, w.dt, st3.T, w.gamma, st3.seed, 40, 2, st3.slab_rate * 40.0,
                    st3.slab_rate, w.rebuild_every, st3.e_rep, None, st3.ekin)
    torch.cuda.synchronize()
    assert ctx3.status() == 0
    assert np.array_equal(a.untag(a.pos), st3.untag(st3.pos))
    assert np.array_equal(a.untag(a.vel), st3.untag(st3.vel))


def test_async_list_renewal_changes_cost_not_results(B):
    """tbsma_set_async: lists re-filtered one step early into the second half of the buffers, beside the gather passes
    that still read the old half, give the same physics as lists renewed ahead of the gather passes; and the list in
    use after the run still covers the cutoff sphere (forces from it match the oracle at the final positions)"""
    w = W.config3(6, seed=13, length=60.0)
    n_steps = 120
    ca, a = run_gpu_md(B, w, n_steps, variant=2, async_inner=True)
    cb, b = run_gpu_md(B, w, n_steps, variant=2, async_inner=False)
    sa, sb = ca.get_stats(), cb.get_stats()
    assert sa["n_replica_builds"] >= sb["n_replica_builds"] >= 4      # asked for 0.03 A earlier: never fewer
    assert ca.status() == 0 and cb.status() == 0
    xa, xb = a.untag(a.pos)[:, :3].astype(np.float64), b.untag(b.pos)[:, :3].astype(np.float64)
    assert traj_rms(xa, xb) <= 1e-4
    md = run_oracle_md(w, n_steps)
    assert traj_rms(xa, md.x) <= TRAJ_RMS
    for ctx, st in ((ca, a), (cb, b)):
        ctx.compute(st.pos, st.force, st.e_rep, None)
        torch.cuda.synchronize()
        x = st.untag(st.pos)
        o = oracle.compute(x[:, :3].astype(np.float64), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi,
                           periodic=w.periodic)
        f = st.untag(st.force)
        err = np.linalg.norm(f[:, :3] - o["f"], axis=1)
        assert np.all(err <= F_ABS + F_REL * np.linalg.norm(o["f"], axis=1))
        assert np.allclose(st.e_rep.cpu().numpy(), o["e_rep"], rtol=E_REL, atol=0)


def test_conditional_graph_node_is_bitwise_identical(B):
    """tbsma_set_graph 2 vs 1: wrapping the cells + candidates chain in an IF node of the captured step changes which
    kernels are launched, not one bit of the results; S = 0.5 forces that chain to run in some steps"""
    w = W.config3(4, seed=17, length=60.0)

    def run(cond):
        ctx = B.make_context(w)
        ctx.set_variant(2)
        ctx.set_outer_skin(0.5)
        ctx.set_graph(True, conditional=cond)
        st = B.DeviceState(w)
        ctx.build_cells(st.pos, st.vel, st.tag)
        ctx.build_neighbors(st.pos, st.vel, st.tag)
        ctx.compute(st.pos, st.force, st.e_rep, None)
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, 100, None, st.slab_rate,
                       0, st.e_rep, None, st.ekin)
        torch.cuda.synchronize()
        assert ctx.status() == 0
        return ctx.get_stats(), st

    sa, a = run(True)
    sb, b = run(False)
    assert sa == sb and sa["n_candidate_builds"] >= 1
    for name in ("pos", "vel", "force"):
        assert np.array_equal(a.untag(getattr(a, name)), b.untag(getattr(b, name))), name


def test_stagger_spreads_the_first_rebuilds(B):
    """tbsma_set_stagger: replicas that start together and share a temperature rebuild in the same few steps; with
    the first threshold scaled per replica the same number of steps sees more, smaller rebuild passes"""
    w = W.config4(16, seed=19)       # sixteen 298 K wires
    n_steps = 30
    ca, a = run_gpu_md(B, w, n_steps, variant=2, stagger=True)
    cb, b = run_gpu_md(B, w, n_steps, variant=2, stagger=False)
    sa, sb = ca.get_stats(), cb.get_stats()
    assert sa["n_build_passes"] > sb["n_build_passes"] >= 1
    assert ca.status() == 0 and cb.status() == 0
    xa, xb = a.untag(a.pos)[:, :3].astype(np.float64), b.untag(b.pos)[:, :3].astype(np.float64)
    assert traj_rms(xa, xb) <= 1e-4


@pytest.mark.parametrize("outer_skin", [0.0, 0.5, 2.0])
def test_candidate_list_radius_changes_cost_not_results(B, outer_skin):
    """tbsma_set_outer_skin: lists filtered from candidates (radius r_cut + skin + S) are the same sets, and the
    trajectory the same bits, for every S; small S forces candidate rebuilds, large S none"""
    w = W.config2(length=60.0)
    n_steps = 150

    def run(S):
        ctx = B.make_context(w)
        ctx.set_variant(2)
        ctx.set_outer_skin(S)
        st = B.DeviceState(w)
        ctx.build_cells(st.pos, st.vel, st.tag)
        ctx.build_neighbors(st.pos, st.vel, st.tag)
        cg, lg = gpu_neighbors(B, ctx, st)
        co, lo = oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
        assert_same_sets(cg, lg, co, lo)
        ctx.compute(st.pos, st.force, st.e_rep, None)
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate,
                       0, st.e_rep, None, st.ekin)
        torch.cuda.synchronize()
        # after the run the list still holds exactly the pairs within r_cut + skin of the positions it was built for
        assert ctx.status() == 0
        return ctx.get_stats(), st

    sa, a = run(outer_skin)
    sb, b = run(2.0)
    assert sa["n_replica_builds"] == sb["n_replica_builds"] >= 5
    if outer_skin == 0.0:
        assert sa["n_candidate_builds"] == sa["n_replica_builds"]
    if outer_skin == 2.0:     # only the relaxation of the as-cut wire ends moves an atom 0.8 A
        assert sa["n_candidate_builds"] <= 2
    # same physics; the slot order (hence the fp32 summation order) depends on when candidates were rebuilt
    xa, xb = a.untag(a.pos)[:, :3].astype(np.float64), b.untag(b.pos)[:, :3].astype(np.float64)
    assert traj_rms(xa, xb) <= 1e-4
    md = run_oracle_md(w, n_steps)
    assert traj_rms(xa, md.x) <= TRAJ_RMS


@pytest.mark.parametrize("outer_skin", [0.6, 2.0])
def test_lists_filtered_from_candidates_are_bit_exact_after_motion(B, outer_skin):
    """rebuild_every = 1 rebuilds every list in every step, so after n steps the list must be exactly the oracle's
    neighbour sets of the FINAL positions -- filtered from candidates collected at step 0 (S = 2.0) or re-collected
    whenever an atom strayed (S = 0.6)"""
    w = W.config3(2, seed=9, length=60.0)         # one 10 K and one 298 K replica
    ctx = B.make_context(w)
    ctx.set_variant(2)
    ctx.set_outer_skin(outer_skin)
    st = B.DeviceState(w)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    n_steps = 120
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate,
                   1, st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    stats = ctx.get_stats()
    assert stats["n_replica_builds"] == w.n_replicas * (n_steps + 1)      # + the build before the run
    if outer_skin == 2.0:
        assert stats["n_candidate_builds"] <= 2 * w.n_replicas
    else:
        assert 0 < stats["n_candidate_builds"] < stats["n_replica_builds"]
    cg, lg = gpu_neighbors(B, ctx, st)
    final = st.untag(st.pos)
    co, lo = oracle.neighbors(final, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert_same_sets(cg, lg, co, lo)
    moved = np.linalg.norm(final[:, :3] - w.pos4[:, :3], axis=1)
    assert moved.max() > 0.15                      # the lists really changed
    assert not np.array_equal(co, oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi,
                                                   w.periodic, max_nb=96)[0])


def test_auto_variant_and_tile_shapes(B):
    """auto picks the shared-memory tiles for wires and the global lists for periodic systems; every
    tile shape gives the same neighbour sets and forces within the bars"""
    _, _ = setup(B, small_bulk(4))
    ctx, st = setup(B, small_bulk(4))
    assert ctx.get_variant() == 1
    w = W.config4(3, seed=5)
    co, lo = oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    o = oracle.compute(w.x64(), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, periodic=w.periodic)
    for tile in [None, (1, 128), (2, 64), (3, 512), (8, 256)]:
        ctx, st = setup(B, w, tile=tile)
        assert ctx.get_variant() == 2
        cg, lg = gpu_neighbors(B, ctx, st)
        assert_same_sets(cg, lg, co, lo)
        ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
        torch.cuda.synchronize()
        assert ctx.status() == 0
        assert_forces(st.untag(st.force)[:, :3].astype(np.float64), o["f"])
        assert np.all(np.abs(st.e_rep.cpu().numpy() - o["e_rep"]) <= E_REL * np.abs(o["e_rep"]))
    bad = B.make_context(small_bulk(4))
    bad.set_variant(2)
    stb = B.DeviceState(small_bulk(4))
    with pytest.raises(B.TbsmaError) as e:       # a periodic axis shorter than three tile cells cannot use the tile variant
        bad.build_cells(stb.pos, stb.vel, stb.tag)
    assert e.value.code == B.EINVAL


def test_philox_noise_matches_oracle(B):
    """free particles (10 A apart, no forces): one step gives v1 = c1 v0 + c2 sigma g, so g is
    recovered from the GPU velocities and compared with the oracle's Philox/Box-Muller."""
    g = np.arange(6) * 10.0
    x = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    n = len(x)
    offs = np.array([0, 100, n], np.int32)
    p4 = W.pack_pos4(x)
    T = np.array([298.0, 10.0], np.float32)
    seed = np.array([0x0123456789ABCDEF, 77], dtype=np.uint64)
    w = W.Workload("free", p4, W.pack_vel4(np.zeros((n, 3)), p4), offs, np.full((2, 3), -5, np.float32),
                   np.full((2, 3), 60, np.float32), np.zeros((2, 3), np.uint8), T, seed, np.zeros(2), gamma=0.05)
    ctx, st = setup(B, w)
    ctx.compute(st.pos, st.force)
    step = (5 << 32) + 12345
    ctx.md_step(st.pos, st.vel, st.force, st.tag, 2.0, st.T, w.gamma, st.seed, step)
    torch.cuda.synchronize()
    v = st.untag(st.vel)[:, :3].astype(np.float64)
    c2 = math.sqrt(1 - math.exp(-2 * w.gamma * 2.0))
    for i in range(n):
        r = 0 if i < 100 else 1
        sig = math.sqrt(KB * float(T[r]) * ACC / MASS)
        gi, _ = oracle.gauss3(int(seed[r]), i - offs[r], step)
        assert np.allclose(v[i] / (c2 * sig), gi, atol=2e-5), i


def test_rebuild_every_cadence_bulk(B):
    w = small_bulk(6)
    ctx, st = run_gpu_md(B, w, 50)
    md = run_oracle_md(w, 50)
    L = float(w.box_hi[0, 0])
    assert traj_rms(st.untag(st.pos)[:, :3].astype(np.float64), md.x, L) <= TRAJ_RMS
    stats = ctx.get_stats()
    # the initial explicit build + the cadence rebuilds at steps 0, 10, 20, 30, 40
    assert stats["n_build_passes"] == 6 and stats["n_replica_builds"] == 6
    assert ctx.status() & B.FLAG_SKIN_VIOLATED == 0
    assert abs(st.e_rep.item() - md.e_rep[0]) <= 5e-6 * abs(md.e_rep[0])


def test_nve_energy_conservation_gpu(B):
    w = W.config1()
    ctx, st = setup(B, w)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    e = []
    with torch.cuda.stream(stream):
        for blk in range(20):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, 2.0, st.T, 0.0, st.seed, blk * 50, 50, None, None, 0,
                       st.e_rep, None, st.ekin)
            stream.synchronize()
            e.append((st.e_rep.item() + st.ekin.item()) / w.n_atoms)
    e = np.array(e)
    assert np.abs(e - e[0]).max() < 3e-5 and abs(e[-4:].mean() - e[:4].mean()) < 5e-6


def test_md_run_host_matches_device_path(B):
    w = W.config2(length=60.0)
    _, st = run_gpu_md(B, w, 30)
    ctx = B.make_context(w)
    pos, vel = w.pos4.copy(), w.vel4.copy()
    force = np.zeros_like(pos)
    tag = np.arange(w.n_atoms, dtype=np.int32)
    e, k = np.zeros(1), np.zeros(1)
    ctx.md_run_host(pos, vel, force, tag, w.dt, w.T, w.gamma, w.seed, 0, 30, None, w.slab_rate, 0, e, None, k)
    out = np.empty_like(pos)
    out[tag] = pos
    assert np.array_equal(out, st.untag(st.pos))
    assert e[0] == pytest.approx(st.e_rep.item(), rel=1e-12) and k[0] == pytest.approx(st.ekin.item(), rel=1e-12)


@pytest.mark.parametrize("which", ["config3", "config4", "config5a", "config5b"])
def test_full_size_sampled_parity(B, which):
    """BASELINE full sizes, in the configuration bench.py times: sampled atoms recomputed one by one
    by the oracle from scratch (brute force over the whole replica)."""
    w = {"config3": W.config3, "config4": W.config4, "config5a": W.config5a, "config5b": W.config5b}[which]()
    ctx, st = setup(B, w)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    rng = np.random.default_rng(0)
    m = 48 if which in ("config3", "config4") else 24
    idx = np.sort(rng.choice(w.n_atoms, m, replace=False))
    s = oracle.compute_sample(w.x64(), w.r_cut, idx, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, periodic=w.periodic)
    fe = st.untag(st.force)
    assert_forces(fe[idx, :3].astype(np.float64), s["f"])
    assert np.abs(fe[idx, 3] - s["e_atom"]).max() < 1e-5
    # properties that hold at any size: momentum conservation per replica, list symmetry via counts
    f = fe[:, :3].astype(np.float64)
    for r in range(0, w.n_replicas, max(1, w.n_replicas // 8)):
        sl = slice(w.offsets[r], w.offsets[r + 1])
        assert np.abs(f[sl].sum(0)).max() < 2e-3
    entries, pairs = ctx.count_pairs(st.pos)
    assert entries % 2 == 0 and pairs % 2 == 0
    # whole-replica energy against the linked-cell oracle for one replica / a 10^6-atom box
    if which in ("config3", "config4"):
        r = 200 if which == "config3" else 1234
        sub = w.take(r, r + 1)
        oc = oracle.compute(sub.x64(), w.r_cut, lo=sub.box_lo, hi=sub.box_hi, cells=True)
        assert abs(st.e_rep[r].item() - oc["e_rep"][0]) <= E_REL * abs(oc["e_rep"][0])
    elif which == "config5b":
        oc = oracle.compute(w.x64(), w.r_cut, lo=w.box_lo, hi=w.box_hi, cells=True)
        assert abs(st.e_rep[0].item() - oc["e_rep"][0]) <= E_REL * abs(oc["e_rep"][0])
        assert_forces(f, oc["f"])
        assert pairs == oc["n_pairs_directed"]
    else:
        oc = oracle.compute(w.x64(), w.r_cut, lo=w.box_lo, hi=w.box_hi, periodic=1, cells=True)
        assert abs(st.e_rep[0].item() - oc["e_rep"][0]) <= E_REL * abs(oc["e_rep"][0])
        assert_forces(f, oc["f"])
        assert pairs == oc["n_pairs_directed"]


def test_full_size_trajectory_in_bench_configuration(B):
    """config 3 at full size with every default bench.py runs with (tile variant, colour placement, staggered first
    rebuilds, asynchronous list renewal beside the gather passes, conditional graph node): 100 steps (the length the
    1e-3 A bound of BASELINE.json's north_star is quoted at), then three replicas
    (a 10 K one, a 298 K one that has rebuilt its list, the last one) are compared with the oracle run of that replica
    ALONE -- positions, velocities, per-replica energies"""
    w = W.config3()
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps)
    assert ctx.status() == 0 and ctx.get_variant() == 2
    stats = ctx.get_stats()
    assert stats["n_replica_builds"] >= 128          # every 298 K replica has renewed its list at least once
    x = st.untag(st.pos)[:, :3].astype(np.float64)
    v = st.untag(st.vel)[:, :3].astype(np.float64)
    e_rep, ekin = st.e_rep.cpu().numpy(), st.ekin.cpu().numpy()
    for r in (5, 200, 255):
        sub = w.take(r, r + 1)
        md = run_oracle_md(sub, n_steps)
        sl = slice(w.offsets[r], w.offsets[r + 1])
        assert traj_rms(x[sl], md.x) <= TRAJ_RMS
        assert np.abs(v[sl] - md.v).max() < 2e-5
        assert abs(e_rep[r] - md.e_rep[0]) <= 10 * E_REL * abs(md.e_rep[0])     # 100 steps of fp32 drift, not one evaluation
        assert abs(ekin[r] - md.ekin_rep[0]) <= 2e-3 * md.ekin_rep[0]


def test_full_size_trajectory_config4_in_bench_configuration(B):
    """config 4 at full size (2048 ragged replicas, 5.4 M atoms, all at 298 K: the persistent gather kernels on a ragged
    tile list with every replica renewing its list), every default of bench.py: 100 steps, then five replicas covering
    the three layer counts are compared with the oracle's run of that replica ALONE"""
    w = W.config4()
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps)
    assert ctx.status() == 0 and ctx.get_variant() == 2
    n_tiles, box, persistent = ctx.get_tiling()
    assert persistent and not box and n_tiles >= 3 * w.n_replicas
    assert ctx.get_stats()["n_replica_builds"] >= 2 * w.n_replicas
    sizes = np.diff(w.offsets)
    assert len(set(sizes)) == 3
    picks = [int(np.nonzero(sizes == n)[0][k]) for n, k in zip(sorted(set(sizes)), (0, -1, 7))] + [1000, w.n_replicas - 1]
    x = st.untag(st.pos)[:, :3].astype(np.float64)
    v = st.untag(st.vel)[:, :3].astype(np.float64)
    e_rep, ekin = st.e_rep.cpu().numpy(), st.ekin.cpu().numpy()
    for r in picks:
        md = run_oracle_md(w.take(r, r + 1), n_steps)
        sl = slice(w.offsets[r], w.offsets[r + 1])
        assert traj_rms(x[sl], md.x) <= TRAJ_RMS
        assert np.abs(v[sl] - md.v).max() < 2e-5
        assert abs(e_rep[r] - md.e_rep[0]) <= 10 * E_REL * abs(md.e_rep[0])
        assert abs(ekin[r] - md.ekin_rep[0]) <= 2e-3 * md.ekin_rep[0]


@pytest.mark.parametrize("name", ["5a", "5b"])
def test_full_size_trajectory_config5_in_bench_configuration(B, name):
    """config 5 at full size with the library's own choices, as bench.py runs it: the 64^3 periodic block (1 048 576 atoms,
    4 394 box tiles) and the 6 nm x 100 nm wire (164 885 atoms, global gather), NVE, lists rebuilt every 10 steps, 100
    steps against the linked-cell oracle: positions, velocities, energy"""
    w = W.config5a() if name == "5a" else W.config5b()
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps)
    assert ctx.status() == 0
    n_tiles, box, _ = ctx.get_tiling()
    assert (ctx.get_variant(), n_tiles, box) == ((2, 4394, True) if name == "5a" else (1, 0, False))
    md = run_oracle_md(w, n_steps)
    L = float(w.box_hi[0, 0] - w.box_lo[0, 0]) if name == "5a" else None
    assert traj_rms(st.untag(st.pos)[:, :3].astype(np.float64), md.x, L) <= TRAJ_RMS
    assert np.abs(st.untag(st.vel)[:, :3].astype(np.float64) - md.v).max() < 2e-5
    assert abs(st.e_rep.item() - md.e_rep[0]) <= 10 * E_REL * abs(md.e_rep[0])


def test_trajectory_ragged_config4_batch_100_steps(B):
    """BASELINE config 4 in small: six replicas of the jittered 3 nm x 6 nm wire (three different layer counts), 298 K
    Langevin + pulling, every bench default on; 100 steps, EVERY replica against the oracle's run of the whole batch
    (north_star: trajectories within 1e-3 A RMS after 100 steps on all five workloads)"""
    w = W.config4(6, seed=35)
    assert len(set(np.diff(w.offsets))) == 3
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps)
    assert ctx.status() == 0 and ctx.get_variant() == 2
    md = run_oracle_md(w, n_steps)
    x = st.untag(st.pos)[:, :3].astype(np.float64)
    v = st.untag(st.vel)[:, :3].astype(np.float64)
    e_rep, ekin = st.e_rep.cpu().numpy(), st.ekin.cpu().numpy()
    for r in range(w.n_replicas):
        sl = slice(w.offsets[r], w.offsets[r + 1])
        assert traj_rms(x[sl], md.x[sl]) <= TRAJ_RMS
        assert np.abs(v[sl] - md.v[sl]).max() < 2e-5
        assert abs(e_rep[r] - md.e_rep[r]) <= 10 * E_REL * abs(md.e_rep[r])
        assert abs(ekin[r] - md.ekin_rep[r]) <= 2e-3 * md.ekin_rep[r]
    pulled = w.flags == 2
    zref = w.vel4[:, 3].astype(np.float64)
    rep = np.searchsorted(w.offsets, np.arange(w.n_atoms), side="right") - 1
    want = (zref + w.slab_rate[rep] * n_steps).astype(np.float32)
    assert np.array_equal(st.untag(st.pos)[pulled, 2], want[pulled])          # placed, to the bit (D:A10)


@pytest.mark.parametrize("variant", [0, 1])
def test_trajectory_thick_wire_config5b_shape_100_steps(B, variant):
    """BASELINE config 5b in small: a 6 nm x 12 nm wire (same cross-section, sigma = 0.05 A start, NVE, list rebuilt
    every 10 steps).  variant 0 = whatever the library picks for a wire this thick, 1 = the global-gather kernels that
    a wire whose layers do not fit a tile falls back to; 100 steps against the oracle."""
    w = W.config5b(length=120.0)
    assert w.rebuild_every == 10
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps, variant=variant)
    assert ctx.status() == 0
    if variant == 1:
        assert ctx.get_variant() == 1
    md = run_oracle_md(w, n_steps)
    assert traj_rms(st.untag(st.pos)[:, :3].astype(np.float64), md.x) <= TRAJ_RMS
    assert np.abs(st.untag(st.vel)[:, :3].astype(np.float64) - md.v).max() < 2e-5
    assert abs(st.e_rep.item() - md.e_rep[0]) <= 10 * E_REL * abs(md.e_rep[0])


def test_trajectory_against_oracle_stepping_with_the_fp32_predicate(B):
    """the oracle stepped with the membership predicate of D:A6 (fp32, the one the kernels use) instead of the fp64
    distance: config 1, 100 steps.  The two oracle runs differ only by pairs within an fp32 ulp of r_cut."""
    w = W.config1()
    n_steps = 100
    ctx, st = run_gpu_md(B, w, n_steps)
    md32 = run_oracle_md(w, n_steps, fp32_pred=True)
    md64 = run_oracle_md(w, n_steps, fp32_pred=False)
    x = st.untag(st.pos)[:, :3].astype(np.float64)
    assert traj_rms(x, md32.x) <= TRAJ_RMS
    assert traj_rms(md32.x, md64.x) <= 1e-6


def test_stress_and_kinetic_tensor_match_oracle(B):
    """tbsma_kinetic_tensor / tbsma_stress (Eq.5 as read in A11) after 30 Langevin steps with grips and pulling: K from
    the same fp32 velocities to rounding, tr K = 2 E_kin of the force pass, sigma = -(W + K) / V against the numpy
    oracle fed with the fp64 oracle's virial of the final positions"""
    from oracle import observables as ob
    w = W.config3(4, seed=23, length=60.0)
    ctx, st = run_gpu_md(B, w, 30, virial=True)
    R = w.n_replicas
    k = torch.full((R, 6), -1.0, dtype=torch.float64, device="cuda")
    sig = torch.zeros(R, 6, dtype=torch.float64, device="cuda")
    n_r = np.diff(w.offsets).astype(np.float64)
    vol = n_r * W.A_LATTICE ** 3 / 4          # one fcc atomic volume per atom, held constant
    d_vol = torch.from_numpy(vol).cuda()
    ctx.kinetic_tensor(st.pos, st.vel, k)
    ctx.stress(st.w_rep, k, d_vol, sig)
    torch.cuda.synchronize()
    v = st.untag(st.vel)[:, :3].astype(np.float64)
    x = st.untag(st.pos)
    K = ob.kinetic_tensor(v, w.flags, w.offsets, oracle.au_params().mass_amu)
    kg = k.cpu().numpy()
    assert np.allclose(kg, K, rtol=1e-11, atol=1e-12)
    assert np.allclose(kg[:, :3].sum(1), 2 * st.ekin.cpu().numpy(), rtol=1e-6)      # the force pass sums E_kin in fp32 terms
    o = oracle.compute(x[:, :3].astype(np.float64), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi,
                       periodic=w.periodic)
    s_ref = ob.stress(o["w_rep"], K, vol)
    sg = sig.cpu().numpy()
    scale = (np.abs(o["w_rep"][:, :3]).sum(1) + n_r * 1e-3) / vol
    assert np.all(np.abs(sg - s_ref) <= 2e-5 * scale[:, None])
    # a stretched wire at 298 K is under tension along its axis: a few GPa
    assert np.all(sg[R // 2:, 2] * ob.EV_PER_A3_IN_GPA > 0)
    # 0 K stress: K = NULL
    ctx.stress(st.w_rep, None, d_vol, sig)
    torch.cuda.synchronize()
    assert np.allclose(sig.cpu().numpy(), -st.w_rep.cpu().numpy() / vol[:, None], rtol=1e-14, atol=0)


@pytest.mark.parametrize("overlap", [1, 2])
def test_overlapped_renewal_waits_for_a_long_filter_pass(B, overlap):
    """512 hot replicas built together and NOT staggered all renew their lists in the same step: the filter pass then
    outlasts both gather passes beside it.  The step must still not swap the list halves before it has finished
    (two streams: join event; programmatic dependent launch: the density pass waits for its primary before it exits).
    Same bits as the kernels one after the other."""
    w = W.config4(512, seed=29)
    n_steps = 30
    ca, a = run_gpu_md(B, w, n_steps, variant=2, overlap=overlap, stagger=False)
    cb, b = run_gpu_md(B, w, n_steps, variant=2, overlap=0, stagger=False)
    sa, sb = ca.get_stats(), cb.get_stats()
    assert sa == sb and sa["n_replica_builds"] >= 512 and sa["n_build_passes"] <= 20     # bunched in a few steps
    assert ca.status() == 0 and cb.status() == 0
    for name in ("pos", "vel", "force"):
        assert np.array_equal(a.untag(getattr(a, name)), b.untag(getattr(b, name))), name


@pytest.mark.parametrize("variant", VARIANTS)
def test_nose_hoover_trajectory_matches_oracle(B, variant):
    """tbsma_set_thermostat(1, tau): the paper's thermostat (reading A17) as B A N A B; two replicas of the same
    wire started at 300 K with targets 150 K and 450 K, 100 steps, against oracle/nose_hoover.py"""
    from oracle.nose_hoover import NoseHooverMD
    base = W.config1()
    n = base.n_atoms
    v = W.maxwell_velocities(n, 300.0, 5, np.ones(n, bool))
    w = W._assemble("nh_2x_wire_3x6nm", [base.x64(), base.x64()], [np.zeros(n, np.int32)] * 2, [v, v], [150.0, 450.0],
                    [1, 2], [0.0, 0.0], 0.0)
    tau, n_steps = 50.0, 100
    ctx, st = setup(B, w, variant=variant)
    ctx.set_thermostat(1, tau)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, 0.0, st.seed, 0, n_steps, None, None, 0, st.e_rep, None,
                   st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    nh = NoseHooverMD(w.x64(), w.v64(), w.flags, w.r_cut, w.T.astype(np.float64), tau, lo=w.box_lo, hi=w.box_hi,
                      offsets=w.offsets)
    for s in range(n_steps):
        nh.step(w.dt)
    xg = st.untag(st.pos)[:, :3].astype(np.float64)
    vg = st.untag(st.vel)[:, :3].astype(np.float64)
    assert traj_rms(xg, nh.x) <= TRAJ_RMS
    assert np.abs(vg - nh.v).max() < 2e-5
    xi, eta = ctx.get_thermostat()
    assert np.allclose(xi, nh.xi, rtol=2e-4, atol=1e-8) and np.allclose(eta, nh.eta, rtol=2e-4, atol=1e-7)
    assert eta[0] > 0 > eta[1]                    # net cooling of the first replica, net heating of the second
    ek = st.ekin.cpu().numpy()
    assert np.allclose(ek, nh.kinetic(), rtol=1e-4)
    # bitwise repeatable (the kinetic energy that drives xi is added in a fixed order), and resumable: 60 steps, state
    # out (pos, vel, force, tag are the caller's; xi, eta through the ABI), a NEW context, state in, 40 steps
    def nh_run(pieces):
        c2, s2 = setup(B, w, variant=variant)
        c2.set_thermostat(1, tau)
        c2.compute(s2.pos, s2.force, s2.e_rep, None)
        torch.cuda.synchronize()
        s0 = 0
        for k, m in enumerate(pieces):
            if k > 0:
                xi2, eta2 = c2.get_thermostat()
                c3 = B.make_context(w, max_neighbors=96)
                c3.set_variant(variant)
                c3.set_thermostat(1, tau)
                c3.build_cells(s2.pos, s2.vel, s2.tag)
                c3.build_neighbors(s2.pos, s2.vel, s2.tag)
                c3.compute(s2.pos, s2.force, s2.e_rep, None)   # the build permuted pos / vel / tag, not the caller's forces
                c3.set_thermostat_state(xi2, eta2)
                torch.cuda.synchronize()
                c2 = c3
            with torch.cuda.stream(stream):
                c2.md_run(s2.pos, s2.vel, s2.force, s2.tag, w.dt, s2.T, 0.0, s2.seed, s0, m, None, None, 0, s2.e_rep, None,
                          s2.ekin)
            torch.cuda.synchronize()
            s0 += m
        return s2.untag(s2.pos), s2.untag(s2.vel), c2.get_thermostat()
    xa, va, (xia, etaa) = nh_run([n_steps])
    assert np.array_equal(xa, st.untag(st.pos)) and np.array_equal(va, st.untag(st.vel))
    assert np.array_equal(xia, xi) and np.array_equal(etaa, eta)
    # resumed in a new context the lists are rebuilt at step 60 (another fp32 summation order): same physics, not same bits
    xb, vb, (xib, etab) = nh_run([60, 40])
    assert np.abs(xb[:, :3] - xa[:, :3]).max() < 1e-4 and np.abs(vb[:, :3] - va[:, :3]).max() < 2e-6
    assert np.allclose(xib, xia, rtol=1e-5, atol=1e-10) and np.allclose(etab, etaa, rtol=1e-5, atol=1e-9)
    # back to Langevin / velocity Verlet: the thermostat state is reset
    ctx.set_thermostat(0)
    assert np.all(ctx.get_thermostat()[0] == 0)


@pytest.mark.parametrize("balance,cell", [(0, 0.0), (1, 0.0), (1, 0.9), (1, 6.0)])
def test_image_placement_changes_cost_not_results(B, balance, cell):
    """tbsma_set_balance: records placed in the tile image in slot order, by the default 2.04 A colour cells, or by
    cells that fit the lattice badly -- the neighbour sets are the oracle's, bit for bit, after the build and after
    60 steps with rebuilds, and the trajectory is the oracle's"""
    w = W.config3(3, seed=31, length=60.0)
    ctx = B.make_context(w)
    ctx.set_variant(2)
    ctx.set_balance(balance, cell)
    st = B.DeviceState(w)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    cg, lg = gpu_neighbors(B, ctx, st)
    co, lo = oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert_same_sets(cg, lg, co, lo)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    n_steps = 60
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate,
                   1, st.e_rep, None, st.ekin)          # rebuild_every = 1: the lists are those of the final positions
    torch.cuda.synchronize()
    assert ctx.status() == 0
    cg, lg = gpu_neighbors(B, ctx, st)
    xf = st.untag(st.pos)
    co, lo = oracle.neighbors(xf, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert_same_sets(cg, lg, co, lo)
    md = run_oracle_md(w, n_steps)
    assert traj_rms(xf[:, :3].astype(np.float64), md.x) <= TRAJ_RMS


def test_long_run_keeps_a_clean_status_word(B):
    """1500 steps of sixteen 24 nm wires at 298 K under tension (about 120 list renewals per replica, the ends relaxing,
    the wire stretching): no list, candidate or tile overflow, no skin violation, nothing non-finite, and the kinetic
    temperature stays at the thermostat's"""
    w = W.config3(16, seed=37)
    w.T[:] = 298.0
    w.vel4[:, :3] = np.concatenate([W.maxwell_velocities(int(n), 298.0, 1000 + r, w.flags[w.offsets[r]:w.offsets[r + 1]] == 0)
                                    for r, n in enumerate(np.diff(w.offsets))]).astype(np.float32)
    ctx, st = run_gpu_md(B, w, 1500)
    assert ctx.status() == 0
    s = ctx.get_stats()
    assert s["n_replica_builds"] > 16 * 60 and s["max_neighbors_seen"] <= 112
    assert bool(torch.isfinite(st.pos).all()) and bool(torch.isfinite(st.vel).all())
    n_dyn = np.array([(w.flags[w.offsets[r]:w.offsets[r + 1]] == 0).sum() for r in range(w.n_replicas)])
    T_kin = 2 * st.ekin.cpu().numpy() / (3 * n_dyn * 8.617333262e-5)
    assert np.all(np.abs(T_kin - 298.0) < 15.0)


# ---- the paper's elongation protocol and the device-side series of its observables ----------------
def _tensile_setup(B, variant, n_rep=3, every=6, n_steps=60, period=7, capacity=16, ramp=True):
    """n_rep short 3 nm wires (config-3 shape: grips at both ends, 10 K and 298 K), BOTH slabs pulled in strokes of
    `period` steps, the target temperature ramped, the series recorded every `every` steps"""
    w = W.config3(n_rep, seed=41, length=60.0)
    ctx, st = setup(B, w, variant=variant)
    R = w.n_replicas
    rate2 = torch.from_numpy(w.slab_rate.copy()).cuda()
    rate1 = torch.from_numpy(-0.5 * w.slab_rate).cuda()
    disp1 = torch.from_numpy(np.linspace(-0.01, -0.03, R)).cuda()
    T_rate = torch.from_numpy(np.linspace(0.05, 0.2, R).astype(np.float32)).cuda() if ramp else None
    L0 = np.array([w.pos4[w.offsets[r]:w.offsets[r + 1], 2].max() - w.pos4[w.offsets[r]:w.offsets[r + 1], 2].min()
                   for r in range(R)], dtype=np.float64)
    vol = np.diff(w.offsets).astype(np.float64) * 4.08 ** 3 / 4
    dev = dict(series=torch.zeros(R * capacity * 4, dtype=torch.float64, device="cuda"),
               count=torch.zeros(R, dtype=torch.int32, device="cuda"),
               rupture=torch.full((R,), -1, dtype=torch.int64, device="cuda"),
               volume=torch.from_numpy(vol).cuda(), L0=torch.from_numpy(L0).cuda(),
               rate2=rate2, rate1=rate1, disp1=disp1, T_rate=T_rate)
    ctx.set_protocol(slab1_disp0=disp1, slab1_rate=rate1, stepwise_period=period, T_rate=T_rate)
    ctx.set_series(every, capacity, dev["series"], dev["count"], dev["rupture"], dev["volume"], dev["L0"])
    return w, ctx, st, dev, L0, vol


@pytest.mark.parametrize("variant", VARIANTS)
def test_two_sided_stroke_pulling_ramp_and_series_match_oracle(B, variant):
    """tbsma_set_protocol + tbsma_set_series: trajectory, slab placement, and every record of the series
    against oracle/protocol.py:TensileMD"""
    from oracle.protocol import TensileMD
    every, n_steps, period, cap = 6, 60, 7, 16
    w, ctx, st, dev, L0, vol = _tensile_setup(B, variant, every=every, n_steps=n_steps, period=period, capacity=cap)
    R = w.n_replicas
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, dev["rate2"], 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    zref = w.vel4[:, 3].astype(np.float64)
    md = oracle.MD(w.x64(), w.v64(), w.flags, w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, cells=True, zref=zref)
    t = TensileMD(md, w.dt, w.T.astype(np.float64), w.gamma, w.seed, 0, 0.0, w.slab_rate, dev["disp1"].cpu().numpy(),
                  -0.5 * w.slab_rate, period=period, T_rate=dev["T_rate"].cpu().numpy().astype(np.float64), every=every,
                  volume=vol, L0=L0)
    for _ in range(n_steps):
        t.step()
    xg = st.untag(st.pos)
    assert traj_rms(xg[:, :3].astype(np.float64), md.x) <= TRAJ_RMS
    for fl in (1, 2):            # both slabs placed to the bit (D:A10)
        assert np.array_equal(xg[w.flags == fl, 2], md.x[w.flags == fl, 2].astype(np.float32))
    assert np.abs(xg[w.flags == 1, 2].astype(np.float64) - zref[w.flags == 1]).max() > 0.009     # the flag-1 slab moved
    count = dev["count"].cpu().numpy()
    assert np.all(count == n_steps // every)
    ser = dev["series"].cpu().numpy().reshape(R, cap, 4)
    for r in range(R):
        ref = np.array(t.series[r])
        got = ser[r, :count[r]]
        assert np.array_equal(got[:, 0], ref[:, 0])                                  # step numbers
        assert np.allclose(got[:, 1], ref[:, 1], rtol=1e-12, atol=1e-15)              # strain (Eq.4)
        assert np.allclose(got[:, 2], ref[:, 2], rtol=2e-4, atol=2e-5 * np.abs(ref[:, 2]).max())   # sigma_zz (Eq.5)
        assert np.allclose(got[:, 3], ref[:, 3], atol=2e-5)                           # largest z gap
    assert np.all(dev["rupture"].cpu().numpy() == -1)
    # the heat map over all replicas: exact counts
    from oracle.protocol import heat_map
    hist = torch.zeros(8 * 6, dtype=torch.int64, device="cuda")
    lo_y, hi_y = float(ser[..., 2].min()) - 1e-3, float(ser[..., 2].max()) + 1e-3
    ctx.series_histogram(dev["series"], dev["count"], cap, 1, 2, -0.001, 0.002, 8, lo_y, hi_y, 6, hist)
    torch.cuda.synchronize()
    xs = np.concatenate([ser[r, :count[r], 1] for r in range(R)])
    ys = np.concatenate([ser[r, :count[r], 2] for r in range(R)])
    assert np.array_equal(hist.cpu().numpy().reshape(6, 8).astype(np.uint64), heat_map(xs, ys, -0.001, 0.002, 8, lo_y, hi_y, 6))
    assert hist.sum().item() > 0
    # switched off again: no further records, the flag-1 slab stays where it is
    ctx.set_series(0)
    ctx.set_protocol()
    z1 = st.untag(st.pos)[w.flags == 1, 2].copy()
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, n_steps, 12, None, None, 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert np.array_equal(dev["count"].cpu().numpy(), count)
    assert np.array_equal(st.untag(st.pos)[w.flags == 1, 2], z1)


def test_notched_paper_wire_under_the_stroke_schedule_matches_oracle(B):
    """the paper's specimen and loading: the 3.1 nm x 20.4 nm wire with its ring notch (8 850 - 27 =
    8 823 atoms), r_cut 5.8 A, buffer 0.29 A, both gripping slabs displaced by +-0.05 A per stroke (here a stroke every 25
    steps instead of every 10 000), 298 K; two wires with their own seeds, 100 steps = four strokes, against
    oracle/protocol.py:TensileMD: trajectory, slabs placed to the bit, every record of the series"""
    from oracle.protocol import TensileMD
    x = W.ring_notch(W.fcc_wire(31.0, 204.0))
    assert len(x) == 8823
    fl = W.grip_flags(x)
    R, every, n_steps, period, cap = 2, 10, 100, 25, 16
    seeds = [83, 89]
    vels = [W.maxwell_velocities(len(x), 298.0, sd, fl == 0) for sd in seeds]
    w = W._assemble("paper_notched_wire_3.1x20.4nm", [x] * R, [fl] * R, vels, [298.0] * R, seeds, [0.05 / period] * R, 1e-3,
                    stretch=1.0)
    w.r_cut, w.skin = 5.8, 0.29
    ctx, st = setup(B, w)
    assert ctx.get_variant() == 2
    rate2 = torch.from_numpy(w.slab_rate.copy()).cuda()
    rate1 = torch.from_numpy(-w.slab_rate).cuda()
    disp1 = torch.zeros(R, dtype=torch.float64, device="cuda")
    L0 = np.full(R, float(x[:, 2].max() - x[:, 2].min()))
    vol = np.full(R, len(x) * 4.0 / 3.0 * math.pi * (2.884 / 2) ** 3)          # hard-sphere volume
    dev = dict(series=torch.zeros(R * cap * 4, dtype=torch.float64, device="cuda"),
               count=torch.zeros(R, dtype=torch.int32, device="cuda"),
               rupture=torch.full((R,), -1, dtype=torch.int64, device="cuda"),
               volume=torch.from_numpy(vol).cuda(), L0=torch.from_numpy(L0).cuda())
    ctx.set_protocol(slab1_disp0=disp1, slab1_rate=rate1, stepwise_period=period, T_rate=None)
    ctx.set_series(every, cap, dev["series"], dev["count"], dev["rupture"], dev["volume"], dev["L0"])
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, rate2, 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    zref = w.vel4[:, 3].astype(np.float64)
    md = oracle.MD(w.x64(), w.v64(), w.flags, w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, cells=True, zref=zref)
    t = TensileMD(md, w.dt, w.T.astype(np.float64), w.gamma, w.seed, 0, 0.0, w.slab_rate, np.zeros(R), -w.slab_rate,
                  period=period, T_rate=None, every=every, volume=vol, L0=L0)
    for _ in range(n_steps):
        t.step()
    xg = st.untag(st.pos)
    assert traj_rms(xg[:, :3].astype(np.float64), md.x) <= TRAJ_RMS
    for f in (1, 2):
        assert np.array_equal(xg[w.flags == f, 2], md.x[w.flags == f, 2].astype(np.float32))
    moved = xg[w.flags == 2, 2].astype(np.float64) - zref[w.flags == 2]
    assert np.allclose(moved, 0.2, atol=1e-5)                     # four strokes of 0.05 A
    count = dev["count"].cpu().numpy()
    assert np.all(count == n_steps // every)
    ser = dev["series"].cpu().numpy().reshape(R, cap, 4)
    for r in range(R):
        ref = np.array(t.series[r])
        got = ser[r, :count[r]]
        assert np.array_equal(got[:, 0], ref[:, 0])
        assert np.allclose(got[:, 1], ref[:, 1], rtol=1e-12, atol=1e-15)
        assert np.allclose(got[:, 2], ref[:, 2], rtol=2e-4, atol=2e-5 * np.abs(ref[:, 2]).max())
        assert np.allclose(got[:, 3], ref[:, 3], atol=2e-5)
    assert np.all(dev["rupture"].cpu().numpy() == -1)


def test_series_detects_a_parted_wire(B):
    """rupture: a wire whose upper half has been moved 8 A up the axis has a gap wider than r_cut: the first
    record reports it, and the recorded gap is the oracle's"""
    from oracle.protocol import largest_gap
    w = W.config3(2, seed=43, length=60.0)
    z = w.pos4[:, 2]
    cut = (z > 1.0) & (np.arange(w.n_atoms) >= w.offsets[1])          # second replica only
    w.pos4[cut, 2] += 8.0
    w.vel4[cut, 3] += 8.0
    w.box_hi[1, 2] += 8.0
    ctx, st = setup(B, w)
    R, cap = 2, 4
    dev = dict(series=torch.zeros(R * cap * 4, dtype=torch.float64, device="cuda"),
               count=torch.zeros(R, dtype=torch.int32, device="cuda"),
               rupture=torch.full((R,), -1, dtype=torch.int64, device="cuda"),
               volume=torch.ones(R, dtype=torch.float64, device="cuda"), L0=torch.full((R,), 60.0, dtype=torch.float64, device="cuda"))
    ctx.set_series(5, cap, dev["series"], dev["count"], dev["rupture"], dev["volume"], dev["L0"])
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 100, 20, None, st.slab_rate, 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    assert np.array_equal(dev["count"].cpu().numpy(), [4, 4])
    rup = dev["rupture"].cpu().numpy()
    assert rup[0] == -1 and rup[1] == 104                               # first record of a run starting at step 100
    ser = dev["series"].cpu().numpy().reshape(R, cap, 4)
    assert np.array_equal(ser[0, :, 0], [104, 109, 114, 119])
    x = st.untag(st.pos)
    assert ser[1, :, 3].min() > w.r_cut and ser[0, :, 3].max() < 3.0
    assert abs(ser[1, -1, 3] - largest_gap(x[w.offsets[1]:, 2])) < 1e-5      # the last record is that of the last step
    with torch.cuda.stream(stream):                                          # capacity reached: recording stops
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 120, 10, None, st.slab_rate, 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert np.array_equal(dev["count"].cpu().numpy(), [4, 4]) and ctx.status() == 0


def test_series_sees_a_gap_that_opens_beyond_the_box(B):
    """the z bins of the series cover the range the atoms occupy at the step of the record, not the box handed to
    tbsma_set_system: a wire whose box ends at z = 20 A, cut at z = 24 A with the top moved 8 A up (everything above the
    box, where fixed bins would put both sides of the gap into the last bin) is reported parted, with the oracle's gap.
    Atoms outside a non-periodic box are legal (edge cells grow, OUT_OF_BOX says so)."""
    from oracle.protocol import largest_gap
    w = W.config3(2, seed=47, length=60.0)
    second = np.arange(w.n_atoms) >= w.offsets[1]
    cut = (w.pos4[:, 2] > 24.0) & second
    w.pos4[cut, 2] += 8.0
    w.vel4[cut, 3] += 8.0
    w.box_hi[1, 2] = 20.0
    ctx, st = setup(B, w, variant=1)
    R, cap = 2, 2
    dev = dict(series=torch.zeros(R * cap * 4, dtype=torch.float64, device="cuda"),
               count=torch.zeros(R, dtype=torch.int32, device="cuda"),
               rupture=torch.full((R,), -1, dtype=torch.int64, device="cuda"),
               volume=torch.ones(R, dtype=torch.float64, device="cuda"), L0=torch.full((R,), 60.0, dtype=torch.float64, device="cuda"))
    ctx.set_series(5, cap, dev["series"], dev["count"], dev["rupture"], dev["volume"], dev["L0"])
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, 10, None, st.slab_rate, 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == B.FLAG_OUT_OF_BOX
    rup = dev["rupture"].cpu().numpy()
    assert rup[0] == -1 and rup[1] == 4
    ser = dev["series"].cpu().numpy().reshape(R, cap, 4)
    x = st.untag(st.pos)
    assert ser[1, :, 3].min() > w.r_cut and ser[0, :, 3].max() < 3.0
    for r in range(R):
        assert abs(ser[r, -1, 3] - largest_gap(x[w.offsets[r]:w.offsets[r + 1], 2])) < 1e-5


def test_box_tiles_keep_up_with_a_compressed_thick_wire(B):
    """the images of box tiles are sized at tbsma_build_cells and cannot grow inside tbsma_md_run, whose cell rebuilds
    re-bin the atoms: a 6 nm x 8 nm wire between grips, compressed by 3 % in 1500 Langevin steps at 298 K (more atoms
    per cell than at the build), must finish with a clean status word and the oracle's forces for its final positions"""
    w = W._replica_batch("thick_wire_6x8nm_gripped", 1, 60.0, 80.0, [298.0], 71)
    L0 = float(w.pos4[:, 2].max() - w.pos4[:, 2].min())
    n_steps = 1500
    w.slab_rate[:] = -0.03 * L0 / n_steps
    ctx, st = run_gpu_md(B, w, n_steps, variant=2, max_nb=136)    # the seventh fcc shell (7.63 A) comes within r_cut + skin
    n_tiles, box, _ = ctx.get_tiling()
    assert box and n_tiles > 1
    assert ctx.status() == 0
    assert ctx.get_stats()["n_candidate_builds"] >= 1          # cells were re-binned on the way
    xf = st.untag(st.pos)
    assert xf[:, 2].max() < w.pos4[:, 2].max() - 0.02 * L0      # it really was compressed
    o = oracle.compute(xf[:, :3].astype(np.float64), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi,
                       periodic=w.periodic)
    assert_forces(st.untag(st.force)[:, :3].astype(np.float64), o["f"])


def z_periodic_wire(ncell=13, radius=15.0, seed=61):
    """a [100] wire periodic along its axis only: ncell cubic cells long (13: 53.04 A = five tile cells of 9.8 A)"""
    a = W.A_LATTICE
    x = W.fcc_bulk(ncell)
    c = 0.5 * ncell * a + 0.25 * a
    x = W.displace(x[(x[:, 0] - c) ** 2 + (x[:, 1] - c) ** 2 < radius ** 2], 0.05, seed)
    x32 = x.astype(np.float32)
    Lf = np.float32(ncell * a)
    x32[:, 2] = np.where(x32[:, 2] < 0, x32[:, 2] + Lf, x32[:, 2])
    x32[:, 2] = np.where(x32[:, 2] >= Lf, x32[:, 2] - Lf, x32[:, 2])
    n = len(x32)
    pos4 = W.pack_pos4(x32, np.zeros(n, np.int32))
    vel4 = W.pack_vel4(np.zeros((n, 3)), pos4)
    lo = np.array([[x32[:, 0].min() - 2, x32[:, 1].min() - 2, 0.0]], np.float32)
    hi = np.array([[x32[:, 0].max() + 2, x32[:, 1].max() + 2, ncell * a]], np.float32)
    return W.Workload(f"z_periodic_wire_{ncell}", pos4, vel4, np.array([0, n], np.int32), lo, hi,
                      np.array([[0, 0, 1]], np.uint8), np.zeros(1, np.float32), np.array([seed], np.uint64), np.zeros(1), 0.0)


@pytest.mark.parametrize("name", ["bulk_10_b2_nc4", "zwire_13_b3_nc5"])
def test_box_tiles_on_a_periodic_axis_of_exactly_b_plus_2_cells_after_drift(B, name):
    """the shortest periodic axis a box of b cells may sit on holds b + 2 cells (TileDesc): the halo of a
    tile is then the whole axis, wrapped at one end.  b = 2 on the four cells of a 40.8 A cube (boxes of 2 x 2 x 1), b = 3
    on the five cells of a 53 A z-periodic wire (boxes of 3 x 3 x 3).  Hot atoms (900 K, NVE) drift across the boundary
    while the cells and candidates of step 0 stay in use (positions are wrapped only when cells are rebuilt), the lists
    being re-filtered in every step: after 120 steps they must be the oracle's sets for the final, unwrapped positions"""
    if name.startswith("bulk"):
        w, tiles = W.config5a(10, seed=67), 16
    else:
        w, tiles = z_periodic_wire(), 2
    w.vel4[:, :3] = W.maxwell_velocities(w.n_atoms, 900.0, 69)
    ctx, st = setup(B, w, max_nb=128, variant=2)      # hot: the seventh fcc shell (7.63 A) reaches into r_cut + skin
    assert ctx.get_tiling()[:2] == (tiles, True)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    n_steps = 120
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, 0.0, st.seed, 0, n_steps, None, None, 1, st.e_rep, None,
                   st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    assert ctx.get_stats()["n_candidate_builds"] == 1           # the cells of step 0 throughout
    final = st.untag(st.pos)
    per = np.nonzero(w.periodic[0])[0]
    out = (final[:, per] < w.box_lo[0, per]) | (final[:, per] >= w.box_hi[0, per])
    assert out.sum() >= 10                                       # atoms beyond the boundary, not wrapped back
    cg, lg = gpu_neighbors(B, ctx, st)
    co, lo = oracle.neighbors(final, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=128)
    assert_same_sets(cg, lg, co, lo)
    o = oracle.compute(final[:, :3].astype(np.float64), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi,
                       periodic=w.periodic)
    assert_forces(st.untag(st.force)[:, :3].astype(np.float64), o["f"])


def test_youngs_modulus_of_the_papers_smallest_wire(B):
    """Table 3: E = 69.6 GPa at 10 K for D0 = 3.1 nm, L0 = 20.4 nm.  Eight such wires (r_cut = 5.8 A, buffer
    0.29 A, Nose-Hoover, both ends pulled, sigma_zz from the device-side series with the hard-sphere volume N 4/3 pi (r0/2)^3,
    P:87) are held for 20 000 steps and then stretched by 2.5 % in 60 000 steps; the slope of the mean stress-strain
    curve between 0.4 % and 2 % strain must be the paper's modulus to within 15 % (measured here: 70.3 GPa).  A loose physics
    check of the whole path (forces, virial, thermostat, protocol, series), not a parity pin."""
    n_rep = 8
    w = W.paper_wire(1, 10.0, n_rep, 7)
    n_at = int(w.offsets[1])
    fl = W.grip_flags(w.pos4[:n_at, :3].astype(np.float64))
    for r in range(n_rep):
        s = slice(w.offsets[r], w.offsets[r + 1])
        w.flags[s] = fl
        w.pos4[s, 3] = fl.astype(np.int32).view(np.float32)
        w.vel4[s, 3] = w.pos4[s, 2]
        w.vel4[s, :3] = np.where((fl != 0)[:, None], 0.0, w.vel4[s, :3])
    ctx = B.make_context(w)
    st = B.DeviceState(w)
    ctx.set_thermostat(1, 100.0)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    L0 = float(w.pos4[:n_at, 2].max() - w.pos4[:n_at, 2].min())
    vol = np.full(n_rep, n_at * 4.0 / 3.0 * math.pi * (2.884 / 2) ** 3)
    eq_steps, pull_steps, every = 20_000, 60_000, 500
    cap = pull_steps // every + 2
    series = torch.zeros(n_rep * cap * 4, dtype=torch.float64, device="cuda")
    count = torch.zeros(n_rep, dtype=torch.int32, device="cuda")
    rupture = torch.full((n_rep,), -1, dtype=torch.int64, device="cuda")
    d_vol, d_L0 = torch.from_numpy(vol).cuda(), torch.full((n_rep,), L0, dtype=torch.float64, device="cuda")
    r2 = torch.full((n_rep,), 0.5 * 0.025 * L0 / pull_steps, dtype=torch.float64, device="cuda")
    r1 = -r2
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, 2.0, st.T, 0.0, st.seed, 0, eq_steps, None, None, 0, st.e_rep, None, st.ekin)
        ctx.set_protocol(slab1_rate=r1)
        ctx.set_series(every, cap, series, count, rupture, d_vol, d_L0)
        ctx.md_run(st.pos, st.vel, st.force, st.tag, 2.0, st.T, 0.0, st.seed, eq_steps, pull_steps, None, r2, 0, st.e_rep,
                   None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    cnt = count.cpu().numpy()
    assert np.all(cnt == pull_steps // every) and np.all(rupture.cpu().numpy() == -1)
    ser = series.cpu().numpy().reshape(n_rep, cap, 4)[:, :cnt[0]]
    eps, sig = ser[0, :, 1], ser[:, :, 2].mean(0) * 160.21766208            # GPa
    assert abs(eps[-1] - 0.025) < 1e-9
    m = (eps > 0.004) & (eps < 0.02)
    E = np.polyfit(eps[m], sig[m], 1)[0]
    assert abs(E - 69.6) < 0.15 * 69.6, E
    T_kin = 2 * st.ekin.cpu().numpy() / (3 * (fl == 0).sum() * KB)
    assert np.all(np.abs(T_kin - 10.0) < 1.0)


# ---- box tiles (thick wires, periodic bulk; tbsma_set_tile_box forces them on thin wires) -------------------------------
BOX_WORKLOADS = ["config1", "config2", "config4_ragged", "bulk_9", "bulk_13", "bulk_18", "thick_wire"]


@pytest.mark.parametrize("name", BOX_WORKLOADS)
def test_box_tiles_lists_forces_energy(B, name):
    """the shared-memory variant with tiles that are boxes of cells (halo wrapped around periodic axes): neighbour sets
    bit for bit, forces, energies and virial against the oracle"""
    w = WORKLOADS[name]()
    ctx, st = setup(B, w, variant=2, box=True)
    assert ctx.get_variant() == 2
    cg, lg = gpu_neighbors(B, ctx, st)
    co, lo = oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert_same_sets(cg, lg, co, lo)
    ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
    torch.cuda.synchronize()
    assert ctx.status() == 0
    o = oracle.compute(w.x64(), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi, periodic=w.periodic)
    fe = st.untag(st.force)
    assert_forces(fe[:, :3].astype(np.float64), o["f"])
    assert np.abs(fe[:, 3] - o["e_atom"]).max() <= 2e-6 * np.abs(o["e_atom"]).max() + 1e-6
    assert np.all(np.abs(st.e_rep.cpu().numpy() - o["e_rep"]) <= E_REL * np.abs(o["e_rep"]))
    scale = np.abs(o["w_rep"][:, :3]).sum(1, keepdims=True) + w.n_atoms / w.n_replicas * 1e-3
    assert np.all(np.abs(st.w_rep.cpu().numpy() - o["w_rep"]) <= 2e-5 * scale)
    n_list, n_cut = ctx.count_pairs(st.pos)
    assert n_list == int(co.sum()) and 0 < n_cut <= n_list


@pytest.mark.parametrize("name", ["config2", "bulk_9", "bulk_13", "thick_wire"])
def test_box_tiles_trajectory_100_steps(B, name):
    """100 steps on box tiles against the oracle: a pulled Langevin wire (lists renewed from their candidates as atoms
    move), periodic bulk and a thick wire with the fixed cadence of BASELINE config 5"""
    w = WORKLOADS[name]()
    n_steps = 100
    ctx, st = setup(B, w, variant=2, box=True)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate,
                   w.rebuild_every, st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0 and ctx.get_variant() == 2
    md = run_oracle_md(w, n_steps)
    L = float(w.box_hi[0, 0] - w.box_lo[0, 0]) if np.any(w.periodic) else None
    assert traj_rms(st.untag(st.pos)[:, :3].astype(np.float64), md.x, L) <= TRAJ_RMS
    assert np.all(np.abs(st.e_rep.cpu().numpy() - md.e_rep) <= 10 * E_REL * np.abs(md.e_rep))
    # and the lists after the motion are the oracle's for the final positions (cadence 1 would force it; here the last
    # rebuild may be a few steps old, so rebuild explicitly)
    ctx.build_cells(st.pos, st.vel, st.tag)
    ctx.build_neighbors(st.pos, st.vel, st.tag)
    cg, lg = gpu_neighbors(B, ctx, st)
    xf = st.untag(st.pos)
    co, lo = oracle.neighbors(xf, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert_same_sets(cg, lg, co, lo)


@pytest.mark.parametrize("name", ["config1", "config2", "config3_small", "config4_ragged"])
def test_fused_step_of_small_batches_is_bitwise_identical(B, name):
    """tbsma_set_fused_step: the whole step of a small batch as one cooperative kernel, the steps
    that renew a list falling back to the separate kernels, gives the bits of the separate kernels throughout: positions,
    velocities, forces, per-replica energies, kinetic energies and virials, rebuild statistics"""
    w = WORKLOADS[name]()
    n_steps = 150

    def run(fused):
        ctx, st = setup(B, w, variant=2)
        ctx.set_fused_step(fused)
        ctx.set_overlap(0)
        ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate, 0,
                       st.e_rep, st.w_rep, st.ekin)
        torch.cuda.synchronize()
        assert ctx.status() == 0
        return ctx, st

    ca, a = run(True)
    cb, b = run(False)
    assert ca.get_stats() == cb.get_stats() and ca.get_stats()["n_replica_builds"] > w.n_replicas
    for nm in ("pos", "vel", "force"):
        assert np.array_equal(a.untag(getattr(a, nm)), b.untag(getattr(b, nm))), nm
    for nm in ("e_rep", "ekin", "w_rep"):
        assert np.array_equal(getattr(a, nm).cpu().numpy(), getattr(b, nm).cpu().numpy()), nm
    assert ca.launch_count() < 0.45 * cb.launch_count()          # one kernel per ordinary step instead of six
    md = run_oracle_md(w, n_steps)
    assert traj_rms(a.untag(a.pos)[:, :3].astype(np.float64), md.x) <= TRAJ_RMS


def test_fused_step_flag_before_the_build_changes_no_bits(B):
    """tbsma_set_fused_step called BEFORE tbsma_build_cells (the other test toggles it afterwards): a batch of 90 tiles
    that fits the fused step only with fewer parts per tile than the automatic split would give is cut the same way
    whether the fused step is on or off, so the per-replica fp64 sums have the same grouping and the same bits"""
    w = W.config4(30, seed=77)
    n_steps = 40

    def run(fused):
        ctx = B.make_context(w)
        ctx.set_variant(2)
        ctx.set_fused_step(fused)
        ctx.set_overlap(0)
        st = B.DeviceState(w)
        ctx.build_cells(st.pos, st.vel, st.tag)
        ctx.build_neighbors(st.pos, st.vel, st.tag)
        ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
        torch.cuda.synchronize()
        first = (st.e_rep.cpu().numpy().copy(), st.w_rep.cpu().numpy().copy())
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate, 0,
                       st.e_rep, st.w_rep, st.ekin)
        torch.cuda.synchronize()
        assert ctx.status() == 0
        return ctx, st, first

    ca, a, fa = run(True)
    cb, b, fb = run(False)
    assert B.lib().tbsma_get_fused_step(ca._h) == 1 and B.lib().tbsma_get_fused_step(cb._h) == 0
    assert np.array_equal(fa[0], fb[0]) and np.array_equal(fa[1], fb[1])
    for nm in ("pos", "vel", "force"):
        assert np.array_equal(a.untag(getattr(a, nm)), b.untag(getattr(b, nm))), nm
    for nm in ("e_rep", "ekin", "w_rep"):
        assert np.array_equal(getattr(a, nm).cpu().numpy(), getattr(b, nm).cpu().numpy()), nm


@pytest.mark.parametrize("depth", [2, 3])
def test_persistent_gather_kernels_on_a_small_batch_match_one_cta_per_tile(B, depth):
    """tbsma_set_gather(2 | 3): the persistent kernels forced onto a batch of a few tiles (every tile cut into parts, the
    units claimed from the global counter, two or three images per CTA), with virial and closing kick: positions,
    velocities and forces bit-identical to one CTA per tile, per-replica sums equal up to their fp64 summation order,
    and the trajectory is the oracle's"""
    w = W.config3(4, seed=51, length=60.0)
    n_steps = 120

    def run(mode):
        ctx = B.make_context(w)
        ctx.set_variant(2)
        ctx.set_gather(mode)
        ctx.set_fused_step(False)
        st = B.DeviceState(w)
        ctx.build_cells(st.pos, st.vel, st.tag)
        ctx.build_neighbors(st.pos, st.vel, st.tag)
        assert ctx.get_tiling()[2] == (mode != 0)
        ctx.compute(st.pos, st.force, st.e_rep, st.w_rep)
        torch.cuda.synchronize()
        e0, w0 = st.e_rep.cpu().numpy().copy(), st.w_rep.cpu().numpy().copy()
        stream = torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(stream):
            ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate, 0,
                       st.e_rep, st.w_rep, st.ekin)
        torch.cuda.synchronize()
        assert ctx.status() == 0
        return ctx, st, e0, w0

    ca, a, ea, wa = run(depth)
    cb, b, eb, wb = run(0)
    assert ca.get_stats() == cb.get_stats()
    for nm in ("pos", "vel", "force"):
        assert np.array_equal(a.untag(getattr(a, nm)), b.untag(getattr(b, nm))), nm
    assert np.allclose(ea, eb, rtol=1e-12) and np.allclose(wa, wb, rtol=1e-11, atol=1e-9)
    for nm in ("e_rep", "ekin", "w_rep"):
        assert np.allclose(getattr(a, nm).cpu().numpy(), getattr(b, nm).cpu().numpy(), rtol=1e-11, atol=1e-9), nm
    md = run_oracle_md(w, n_steps)
    assert traj_rms(a.untag(a.pos)[:, :3].astype(np.float64), md.x) <= TRAJ_RMS
    assert np.all(np.abs(a.e_rep.cpu().numpy() - md.e_rep) <= 10 * E_REL * np.abs(md.e_rep))


def test_mixed_batch_of_layer_and_box_tiles(B):
    """one batch holding a thin wire (cut into layer tiles), a 6 nm wire (its layers do not fit an image: box tiles) and a
    second thin wire: lists bit for bit, forces and energies against the oracle, and a 60-step Langevin trajectory with the
    lists renewed on the way; each replica's trajectory is the one it has alone (tiles are chosen per replica)"""
    thin = W.displace(W.fcc_wire(30.0, 60.0), 0.05, 61)
    thick = W.displace(W.fcc_wire(60.0, 70.0), 0.05, 62)
    thin2 = W.displace(W.fcc_wire(30.0, 80.0), 0.05, 63)
    wires = [thin, thick, thin2]
    flags = [np.zeros(len(x), np.int32) for x in wires]
    vels = [W.maxwell_velocities(len(x), 200.0, 70 + k, f == 0) for k, (x, f) in enumerate(zip(wires, flags))]
    w = W._assemble("mixed_thin_thick_thin", wires, flags, vels, [200.0] * 3, [5, 6, 7], [0.0] * 3, 1e-3)
    ctx, st = setup(B, w, variant=2, stagger=False)
    n_tiles, box, persistent = ctx.get_tiling()
    assert box and not persistent and n_tiles > 6
    cg, lg = gpu_neighbors(B, ctx, st)
    co, lo = oracle.neighbors(w.pos4, w.r_cut + w.skin, w.offsets, w.box_lo, w.box_hi, w.periodic, max_nb=96)
    assert_same_sets(cg, lg, co, lo)
    ctx.compute(st.pos, st.force, st.e_rep, None)
    torch.cuda.synchronize()
    o = oracle.compute(w.x64(), w.r_cut, offsets=w.offsets, lo=w.box_lo, hi=w.box_hi)
    assert_forces(st.untag(st.force)[:, :3].astype(np.float64), o["f"])
    assert np.all(np.abs(st.e_rep.cpu().numpy() - o["e_rep"]) <= E_REL * np.abs(o["e_rep"]))
    n_steps = 60
    stream = torch.cuda.Stream()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(stream):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, 0, n_steps, None, st.slab_rate, 0,
                   st.e_rep, None, st.ekin)
    torch.cuda.synchronize()
    assert ctx.status() == 0 and ctx.get_stats()["n_replica_builds"] > 3
    md = run_oracle_md(w, n_steps)
    xg = st.untag(st.pos)
    assert traj_rms(xg[:, :3].astype(np.float64), md.x) <= TRAJ_RMS
    # the thin wire alone is cut into the same tiles: same bits
    single = w.take(0, 1)
    _, ss = run_gpu_md(B, single, n_steps, variant=2, stagger=False)
    assert np.array_equal(xg[:w.offsets[1]], ss.untag(ss.pos))
