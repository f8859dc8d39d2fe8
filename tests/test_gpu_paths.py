"""GPU: the alternative kernel paths of libdwf agree with each other (every path is also compared with the
oracle in test_gpu_parity.py / test_gpu_fullsize.py through whichever path is the default).

  * tiled persistent stencil (dwf_tile.cuh)  vs  generic stencil (dwf_hop.cuh)      DWF_NO_TILE=1
  * Schur K1 with the fused M_oo^-1 epilogue vs  separate mooinv_kernel            DWF_NO_FUSE_MOOINV=1
  * CG enqueued on the stream                vs  CG captured into a CUDA graph     DWF_CG_GRAPH=1
  * 16- / 32- / 64-site tiles of the tiled stencil (small lattices default to 16)   DWF_TILE=bx,by,bz,bt
  * dynamic item assignment                  vs  static round robin                DWF_NO_DYN=1
  * one rhs-major launch per batch of rhs    vs  one launch per rhs                DWF_RHS_LOOP=1
  * literal Chebyshev step aH(Ht) - bt       vs  factored a(H - c)(H + c)t         DWF_CHEB_FACTORED=1
"""
import numpy as np
import pytest

import dwf_inputs as gen
from gpu_util import M5, Rig, rel_l2

pytestmark = pytest.mark.gpu

from paper_2103_05034_b200 import DWF_DAGGER, DWF_DDW, DWF_DHOP, DWF_HDW, DWF_SCHUR_EO  # noqa: E402


@pytest.mark.parametrize("prec,L,Ls,nrhs", [("f32", (8, 8, 4, 4), 16, 3), ("f64", (8, 4, 4, 4), 16, 2), ("f32", (8, 4, 4, 8), 24, 2)])
def test_tiled_vs_generic(oracle, monkeypatch, prec, L, Ls, nrhs):
    mass = 0.03
    tol = 1e-12 if prec == "f64" else 2e-6
    psi = None
    outs = {}
    for tag, env in (("tiled", None), ("generic", "1")):
        if env:
            monkeypatch.setenv("DWF_NO_TILE", env)
        rig = Rig(L, Ls, prec, mass, seed_U=31, ws_nrhs=nrhs)
        if psi is None:
            psi = rig.spinor(nrhs, 32)
        pe = gen.keep_parity(psi, L, 0)
        outs[tag] = [rig.apply(DWF_DHOP, psi), rig.apply(DWF_DDW, psi), rig.apply(DWF_HDW, psi), rig.apply(DWF_DDW | DWF_DAGGER, psi),
                     rig.apply(DWF_SCHUR_EO, pe, half=True), rig.apply(DWF_SCHUR_EO | DWF_DAGGER, pe, half=True)]
        cheb = rig.d.field(nrhs)
        rig.d.chebyshev(5, 0.01, 70.0, rig.native(psi), cheb, nrhs)
        outs[tag].append(rig.canonical(cheb, nrhs))
    for a, b in zip(outs["tiled"], outs["generic"]):
        assert rel_l2(a, b) < tol
    # and one of them against the oracle, so that the pair is anchored
    assert rel_l2(outs["generic"][1], oracle.ddw(rig.U, psi, M5, mass)) < (1e-12 if prec == "f64" else 1e-5)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_fused_mooinv_vs_separate(monkeypatch, prec):
    L, Ls, mass, nrhs = (8, 4, 8, 4), 16, 0.01, 2
    rig = Rig(L, Ls, prec, mass, seed_U=41, ws_nrhs=nrhs)
    pe = gen.keep_parity(rig.spinor(nrhs, 42), L, 0)
    fused = [rig.apply(DWF_SCHUR_EO, pe, half=True), rig.apply(DWF_SCHUR_EO | DWF_DAGGER, pe, half=True)]
    monkeypatch.setenv("DWF_NO_FUSE_MOOINV", "1")                     # read at dwf_create: a second handle takes the unfused path
    rig2 = Rig(L, Ls, prec, mass, seed_U=41, ws_nrhs=nrhs)
    l0 = rig2.d.launch_count()
    sep = [rig2.apply(DWF_SCHUR_EO, pe, half=True), rig2.apply(DWF_SCHUR_EO | DWF_DAGGER, pe, half=True)]
    assert rig2.d.launch_count() - l0 == 2 * (1 + (1 + 1 + 1) + 1)         # import, K1 (one rhs-major launch for the batch) + M_oo^-1 + K2, export
    for a, b in zip(fused, sep):
        assert np.array_equal(a, b)                   # same arithmetic in the same order: bit identical


def test_cg_graph_vs_stream(monkeypatch):
    """The CG solve enqueued kernel by kernel (DWF_CG_GRAPH=0) and as one CUDA graph kept instantiated in the handle (the default at
    this launch-bound size; DWF_CG_GRAPH=1 forces it): bit identical, on a cache miss, on a hit, and after the arguments changed."""
    L, Ls, mass = (8, 8, 8, 8), 16, 0.01
    monkeypatch.setenv("DWF_CG_GRAPH", "0")                           # read at dwf_create
    rig = Rig(L, Ls, "f32", mass, seed_U=1001, ws_nrhs=1)
    b = rig.native(gen.keep_parity(rig.spinor(1, 2001), L, 0), 0)
    x1 = rig.d.field(1, half=True, zero=True)
    l0 = rig.d.launch_count()
    h1 = rig.d.cg_schur(b, x1, 20)
    n_stream = rig.d.launch_count() - l0
    for env in ("1", None):
        if env is None:
            monkeypatch.delenv("DWF_CG_GRAPH")
        else:
            monkeypatch.setenv("DWF_CG_GRAPH", env)
        rig2 = Rig(L, Ls, "f32", mass, seed_U=1001, ws_nrhs=1)
        x2 = rig2.d.field(1, half=True, zero=True)
        l0 = rig2.d.launch_count()
        h2 = rig2.d.cg_schur(b, x2, 20)                               # miss: capture + instantiate + launch
        assert rig2.d.launch_count() - l0 == n_stream                 # the graph's kernels are counted once, when it runs
        assert h1 == h2 and bool((x1 == x2).all())                    # deterministic reductions: bit identical
        x2.zero_()
        assert rig2.d.cg_schur(b, x2, 20) == h1 and bool((x1 == x2).all())     # hit: the kept graph is re-launched
        x3 = rig2.d.field(1, half=True, zero=True)
        assert rig2.d.cg_schur(b, x3, 20) == h1 and bool((x1 == x3).all())     # other x: re-captured
        h10 = rig2.d.cg_schur(b, x3.zero_(), 10)                      # other iteration count: re-captured
        assert h10 == h1[:11]


def test_tile_sizes_agree(oracle, monkeypatch):
    """fp32, Ls 16: lattices with fewer than two 32-site tiles per SM default to 16-site tiles (dwf_api.cu build_tables); the
    32-site geometry (the production one at 16^3x32) and the 64-site one are forced through DWF_TILE.  The per-site arithmetic
    does not depend on the tile shape: operator results are bit identical; the CG residual history (reduction order differs)
    agrees to rounding; the default is anchored to the oracle."""
    L, Ls, mass, nrhs = (8, 8, 8, 8), 16, 0.01, 2
    outs, hists = {}, {}
    psi = None
    for tag, env in (("default", None), ("ts32", "4,4,2,2"), ("ts64", "4,4,4,2"), ("ts16", "4,2,2,2")):
        if env:
            monkeypatch.setenv("DWF_TILE", env)
        rig = Rig(L, Ls, "f32", mass, seed_U=51, ws_nrhs=nrhs)
        if psi is None:
            psi = rig.spinor(nrhs, 52)
        pe = gen.keep_parity(psi, L, 0)
        outs[tag] = [rig.apply(DWF_DDW, psi), rig.apply(DWF_HDW, psi), rig.apply(DWF_DDW | DWF_DAGGER, psi),
                     rig.apply(DWF_SCHUR_EO, pe, half=True), rig.apply(DWF_SCHUR_EO | DWF_DAGGER, pe, half=True)]
        cheb = rig.d.field(nrhs)
        rig.d.chebyshev(4, 0.01, 70.0, rig.native(psi), cheb, nrhs)
        outs[tag].append(rig.canonical(cheb, nrhs))
        b = rig.native(gen.keep_parity(psi[:1], L, 0), 0)
        hists[tag] = np.array(rig.d.cg_schur(b, rig.d.field(1, half=True, zero=True), 12))
    assert np.array_equal(outs["default"][0], outs["ts16"][0])          # the default IS the 16-site geometry at this size
    for tag in ("ts32", "ts64", "ts16"):
        for a, b in zip(outs["default"], outs[tag]):
            assert np.array_equal(a, b), tag
        assert np.max(np.abs(hists[tag] - hists["default"]) / hists["default"]) < 1e-5, tag
    assert rel_l2(outs["default"][0], oracle.ddw(rig.U, psi, M5, mass)) < 1e-5
    assert rel_l2(outs["default"][3], oracle.mpc(rig.U, gen.keep_parity(psi, L, 0), M5, mass)) < 1e-5


@pytest.mark.parametrize("prec,tile", [("f32", None), ("f32", "4,4,2,2"), ("f64", None)])
def test_repeatable_bit_for_bit(monkeypatch, prec, tile):
    """The persistent kernel hands its shared-memory buffers over through mbarriers and an atomic counter: a race there would
    show up as run-to-run differences.  30 applies of H_DW (+ the Chebyshev pair, + the fused Schur) on one input at a size with
    many work items per CTA must be bit identical."""
    import torch
    from paper_2103_05034_b200 import DWF_SCHUR_EO
    L, Ls, nrhs = (16, 16, 8, 8), 16, 2
    if tile:
        monkeypatch.setenv("DWF_TILE", tile)              # the 32-site geometry of the bench lattice (this lattice defaults to 16)
    rig = Rig(L, Ls, prec, 0.01, seed_U=81, ws_nrhs=nrhs)
    g = torch.Generator(device="cuda"); g.manual_seed(82)
    x = rig.d.field(nrhs).normal_(generator=g)
    ref_h, ref_c, ref_s = rig.d.field(nrhs), rig.d.field(nrhs), rig.d.field(nrhs, half=True)
    rig.d.apply(DWF_HDW, x, ref_h, nrhs)
    rig.d.chebyshev(3, 0.01, 70.0, x, ref_c, nrhs)
    xe = x[: ref_s.numel()].clone()
    rig.d.apply(DWF_SCHUR_EO, xe, ref_s, nrhs)
    for _ in range(30):
        y, c, s = rig.d.field(nrhs), rig.d.field(nrhs), rig.d.field(nrhs, half=True)
        rig.d.apply(DWF_HDW, x, y, nrhs)
        rig.d.chebyshev(3, 0.01, 70.0, x, c, nrhs)
        rig.d.apply(DWF_SCHUR_EO, xe, s, nrhs)
        assert torch.equal(y, ref_h) and torch.equal(c, ref_c) and torch.equal(s, ref_s)


def test_dynamic_vs_static_assignment_and_batch_vs_loop(monkeypatch):
    """At a size where the tiled kernel hands items out dynamically (more than two items per CTA), no result may depend on which CTA
    computed an item or on how the right-hand sides were cut into launches: operators, Chebyshev and the CG history (fused norms:
    one partial per (item, warp), summed in index order) are bit identical across DWF_NO_DYN / DWF_RHS_LOOP and across repeats."""
    import torch
    L, Ls, nrhs = (16, 16, 16, 16), 16, 3
    res = {}
    for tag, env in (("default", {}), ("static", {"DWF_NO_DYN": "1"}), ("loop", {"DWF_RHS_LOOP": "1"})):
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        rig = Rig(L, Ls, "f32", 0.01, seed_U=61, ws_nrhs=nrhs)
        for k in env:
            monkeypatch.delenv(k)
        g = torch.Generator(device="cuda"); g.manual_seed(62)
        x = rig.d.field(nrhs).normal_(generator=g)
        y, c, se = rig.d.field(nrhs), rig.d.field(nrhs), rig.d.field(nrhs, half=True)
        l0 = rig.d.launch_count()
        rig.d.apply(DWF_DDW, x, y, nrhs)
        n_apply = rig.d.launch_count() - l0
        rig.d.chebyshev(3, 0.01, 70.0, x, c, nrhs)
        xe = x[: se.numel()].clone()
        rig.d.apply(DWF_SCHUR_EO, xe, se, nrhs)
        b = xe[: xe.numel() // nrhs].clone()
        hists, sols = [], []
        for _ in range(3 if tag == "default" else 1):
            xs = rig.d.field(1, half=True, zero=True)
            hists.append(rig.d.cg_schur(b, xs, 6)); sols.append(xs)
        assert all(h == hists[0] for h in hists) and all(bool((s_ == sols[0]).all()) for s_ in sols)
        res[tag] = (y, c, se, hists[0], sols[0], n_apply)
    assert res["default"][5] == 1 and res["loop"][5] == nrhs           # one launch for the batch / one per rhs
    for tag in ("static", "loop"):
        for a, b_ in zip(res["default"][:3], res[tag][:3]):
            assert torch.equal(a, b_), tag
        assert res[tag][3] == res["default"][3] and torch.equal(res[tag][4], res["default"][4]), tag
    # (the default path is compared with the oracle at this kernel geometry -- 32-site tiles, dynamic assignment, batch launches -- by
    # tests/test_gpu_fullsize.py)


@pytest.mark.parametrize("prec,L,Ls", [("f32", (8, 8, 4, 4), 16), ("f64", (8, 4, 4, 4), 16), ("f32", (6, 4, 4, 4), 8)])
def test_chebyshev_factored_step(oracle, monkeypatch, prec, L, Ls):
    """DWF_CHEB_FACTORED=1: alpha H^2 - beta applied as alpha (H - c)(H + c), c = sqrt(beta/alpha), the shift fused into the
    Gamma5 epilogue (tiled and generic kernel).  Same polynomial: against the oracle at the tolerances of the literal form,
    and against the literal form itself."""
    mass, nrhs = 0.01, 2
    tol = {"f32": 1e-4, "f64": 1e-11}[prec]
    outs = {}
    for tag in ("literal", "factored"):
        if tag == "factored":
            monkeypatch.setenv("DWF_CHEB_FACTORED", "1")
        rig = Rig(L, Ls, prec, mass, seed_U=71, ws_nrhs=nrhs)
        psi = rig.spinor(nrhs, 72)
        res = []
        for order in (1, 2, 7, 64):
            out = rig.d.field(nrhs)
            rig.d.chebyshev(order, 0.01, 70.0, rig.native(psi), out, nrhs)
            res.append(rig.canonical(out, nrhs))
        outs[tag] = res
    for order, a, b in zip((1, 2, 7, 64), outs["literal"], outs["factored"]):
        want = oracle.chebyshev(rig.U, psi, M5, mass, order, 0.01, 70.0)
        assert rel_l2(b, want) < tol, order
        assert rel_l2(a, want) < tol, order
        assert rel_l2(a, b) < tol, order
