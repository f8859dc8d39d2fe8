"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times.

configs[2]/[3] (16^3 x 32 x 16): the oracle computes whole right-hand sides one by one, so for
nrhs = 12 / 48 / 24 a SAMPLE of right-hand sides is compared (every rhs is an independent unit).
configs[4] (48^3 x 96 x 24, 24.5 GB per vector): sampled-site parity through the oracle's site-list
mode plus oracle-free invariants for the 100 CG iterations.
"""
import numpy as np
import pytest
import torch

import dwf_inputs as gen
from gpu_util import M5, TOL_APPLY, TOL_CHEB, Rig, rel_l2

pytestmark = pytest.mark.gpu

from paper_2103_05034_b200 import DWF_DDW, DWF_F32, DWF_HDW, DWF_SCHUR_EO, DWF_DAGGER, Dwf  # noqa: E402

L2 = (16, 16, 16, 32)


def _batch_with_samples(rig, nrhs, seed, sample):
    """Canonical device batch of nrhs fields: the sampled rhs are the seeded numpy fields (seed + 100 r),
    the others are filled by torch's seeded generator (they only have to be there)."""
    g = torch.Generator(device="cuda"); g.manual_seed(seed)
    rdt = torch.float32 if rig.prec == "f32" else torch.float64
    can = torch.view_as_complex(torch.randn(rig.d.canonical_shape(nrhs) + (2,), generator=g, device="cuda", dtype=rdt))
    fields = {}
    for r in sample:
        f = gen.round_to_precision(gen.spinor_gaussian(rig.L, rig.Ls, 1, seed + 100 * r), rig.prec)
        fields[r] = f
        can[r] = rig.to_dev(f)[0]
    return can.contiguous(), fields


@pytest.mark.parametrize("prec,nrhs,sample", [("f32", 1, [0]), ("f64", 1, [0]), ("f32", 12, [0, 11]), ("f64", 12, [5]),
                                              ("f32", 48, [0, 23, 47]), ("f64", 48, [7, 47])])
def test_config2_ddw_hdw(oracle, prec, nrhs, sample):
    rig = Rig(L2, 16, prec, 0.01, seed_U=1002)
    can, fields = _batch_with_samples(rig, nrhs, 2002, sample)
    x = rig.d.import_(can)
    del can
    y = rig.d.field(nrhs)
    for op, ref in ((DWF_DDW, lambda f: oracle.ddw(rig.U, f, M5, 0.01)), (DWF_HDW, lambda f: oracle.hdw(rig.U, f, M5, 0.01))):
        rig.d.apply(op, x, y, nrhs)
        out = rig.d.export(y, nrhs)
        for r in sample:
            got = out[r:r + 1].cpu().numpy().astype(np.complex128)
            assert rel_l2(got, ref(fields[r])) < TOL_APPLY[prec], (op, r)
        del out


def test_config3_chebyshev_order64_24vec(oracle):
    rig = Rig(L2, 16, "f32", 0.01, seed_U=1002, ws_nrhs=24)
    sample = [17]
    can, fields = _batch_with_samples(rig, 24, 2003, sample)
    x = rig.d.import_(can)
    del can
    out = rig.d.field(24)
    rig.d.chebyshev(64, 0.01, 70.0, x, out, 24)
    res = rig.d.export(out, 24)
    for r in sample:
        want = oracle.chebyshev(rig.U, fields[r], M5, 0.01, 64, 0.01, 70.0)
        got = res[r:r + 1].cpu().numpy().astype(np.complex128)
        assert rel_l2(got, want) < TOL_CHEB["f32"]
        ratio = np.linalg.norm(got) / np.linalg.norm(fields[r])
        assert 0.6 < ratio < 0.8                                     # |T_64| <= 1 on the spectrum: ~1/sqrt 2
    # oracle-free identity on every vector: T_2n(X) eta = 2 T_n(X) T_n(X) eta - eta (here n = 8)
    t8, t8t8, t16 = rig.d.field(24), rig.d.field(24), rig.d.field(24)
    rig.d.chebyshev(8, 0.01, 70.0, x, t8, 24)
    rig.d.chebyshev(8, 0.01, 70.0, t8, t8t8, 24)
    rig.d.chebyshev(16, 0.01, 70.0, x, t16, 24)
    lhs = 2.0 * t8t8 - x
    num = rig.d.norm2(lhs - t16, 24)
    den = rig.d.norm2(t16, 24)
    assert max(np.sqrt(n / d) for n, d in zip(num, den)) < 2e-5


# ---------------------------------------------------------------------------------- configs[4]
L4 = (48, 48, 48, 96)
LS4, MASS4 = 24, 0.00078


def _sample_sites(L, n_random, seed):
    Lx, Ly, Lz, Lt = L
    rng = np.random.default_rng(seed)
    sites = [tuple(rng.integers(0, L[i]) for i in range(4)) for _ in range(n_random)]
    sites += [(x, y, z, t) for x in (0, Lx - 1) for y in (0, Ly - 1) for z in (0, Lz - 1) for t in (0, Lt - 1)]   # 16 corners
    for mu in range(4):                                              # 64 sites on each of the 8 boundary faces
        for edge in (0, L[mu] - 1):
            for _ in range(64):
                c = [int(rng.integers(0, L[i])) for i in range(4)]
                c[mu] = edge
                sites.append(tuple(c))
    sites += [(Lx - 1 - i % Lx, Ly - 1 - (i // Lx) % Ly, Lz - 1, Lt - 1) for i in range(64)]   # last sites in index order
    return np.array(sorted(set(sites)), dtype=np.int64)


def _gather_two_hop(L, psi, U, st):
    """Two-hop neighbourhoods of the even sites st[n,4] (device) in the layout oracle.mpc_sites expects: indexing only."""
    dev = st.device
    n, Ls = st.shape[0], psi.shape[1]
    Lt_ = torch.tensor(L, device=dev)

    def fetch_psi(c):
        return psi[0][:, c[:, 3], c[:, 2], c[:, 1], c[:, 0]].permute(1, 0, 2, 3).cpu().numpy().astype(np.complex128)

    def fetch_link(mu, c):
        return U[mu][c[:, 3], c[:, 2], c[:, 1], c[:, 0]].cpu().numpy().astype(np.complex128)
    self_ = fetch_psi(st)
    nbr2 = np.zeros((n, 8, 8, Ls, 4, 3), dtype=np.complex128)
    links1 = np.zeros((n, 8, 3, 3), dtype=np.complex128)
    links2 = np.zeros((n, 8, 8, 3, 3), dtype=np.complex128)
    for mu in range(4):
        for j, d in enumerate((+1, -1)):
            y = st.clone(); y[:, mu] = (y[:, mu] + d) % Lt_[mu]
            links1[:, 2 * mu + j] = fetch_link(mu, st if d > 0 else y)
            for nu in range(4):
                for k, e in enumerate((+1, -1)):
                    z = y.clone(); z[:, nu] = (z[:, nu] + e) % Lt_[nu]
                    nbr2[:, 2 * mu + j, 2 * nu + k] = fetch_psi(z)
                    links2[:, 2 * mu + j, 2 * nu + k] = fetch_link(nu, y if e > 0 else z)
    return self_, nbr2, links1, links2


def test_config4_ddw_sampled_and_cg_invariants(oracle):
    import gc
    gc.collect(); torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 150e9:
        pytest.skip("needs ~150 GB of device memory")
    dev = torch.device("cuda")
    d = Dwf(L4, LS4, M5, MASS4, DWF_F32)
    U = gen.gauge_random_torch(L4, 1004, dev, torch.complex64)
    d.set_gauge(U)
    psi = gen.spinor_gaussian_torch(L4, LS4, 1, 2004, dev, torch.complex64)
    x = d.import_(psi)
    y = d.field(1)
    d.apply(DWF_DDW, x, y, 1)
    out = d.export(y, 1)
    del y
    # ---- gather neighbourhoods of the sampled sites and evaluate the definition in fp64 on the host
    sites = _sample_sites(L4, 4096, 4)
    n = len(sites)
    nbr = np.zeros((n, 9, LS4, 4, 3), dtype=np.complex128)
    links = np.zeros((n, 8, 3, 3), dtype=np.complex128)
    st = torch.from_numpy(sites).to(dev)
    def fetch_psi(c):   # c: [n,4] device int64 -> [n, Ls, 4, 3]
        return psi[0][:, c[:, 3], c[:, 2], c[:, 1], c[:, 0]].permute(1, 0, 2, 3).cpu().numpy().astype(np.complex128)
    nbr[:, 0] = fetch_psi(st)
    Lt_ = torch.tensor(L4, device=dev)
    for mu in range(4):
        for j, dirn in enumerate((+1, -1)):
            c = st.clone(); c[:, mu] = (c[:, mu] + dirn) % Lt_[mu]
            nbr[:, 1 + 2 * mu + j] = fetch_psi(c)
            src = st if dirn > 0 else c                          # U_mu(x) or U_mu(x - mu)
            links[:, 2 * mu + j] = U[mu][src[:, 3], src[:, 2], src[:, 1], src[:, 0]].cpu().numpy().astype(np.complex128)
    want = oracle.ddw_sites(L4, LS4, M5, MASS4, sites.astype(np.int32), nbr, links)
    got = out[0][:, st[:, 3], st[:, 2], st[:, 1], st[:, 0]].permute(1, 0, 2, 3).cpu().numpy().astype(np.complex128)
    err = np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel())
    assert err < TOL_APPLY["f32"], err
    worst = np.max(np.linalg.norm((got - want).reshape(n, -1), axis=1) / np.linalg.norm(want.reshape(n, -1), axis=1))
    assert worst < 10 * TOL_APPLY["f32"], worst
    del out
    # ---- the Schur operator and its adjoint at sampled EVEN sites against the definition (Table V):
    # the Ls = 24 tile kernel with the fused closed-form M_oo^-1 and > 2^31 element offsets versus generic elimination on the host
    d.set_workspace(1, half_fields=1)
    hb = d.field_bytes(1, half=True) // 4
    ev = _sample_sites(L4, 8600, 5)
    ev = ev[ev.sum(axis=1) % 2 == 0]
    assert len(ev) >= 4096
    ste = torch.from_numpy(ev).to(dev)
    nb2 = _gather_two_hop(L4, psi, U, ste)
    w = d.field(1, half=True)
    for op, dag in ((DWF_SCHUR_EO, False), (DWF_SCHUR_EO | DWF_DAGGER, True)):
        d.apply(op, x[:hb], w, 1)
        can = d.export(w, 1, parity=0)
        got = can[0][:, ste[:, 3], ste[:, 2], ste[:, 1], ste[:, 0]].permute(1, 0, 2, 3).cpu().numpy().astype(np.complex128)
        del can
        want = oracle.mpc_sites(L4, LS4, M5, MASS4, ev.astype(np.int32), *nb2, dagger=dag)
        err = np.linalg.norm((got - want).ravel()) / np.linalg.norm(want.ravel())
        assert err < TOL_APPLY["f32"], (dag, err)
        worst = np.max(np.linalg.norm((got - want).reshape(len(ev), -1), axis=1) / np.linalg.norm(want.reshape(len(ev), -1), axis=1))
        assert worst < 10 * TOL_APPLY["f32"], (dag, worst)
    del w, nb2
    # ---- hermiticity at full size (oracle-free): <a, H b> = <H a, b>
    b2 = torch.roll(x, 12345)
    Ha, Hb = d.field(1), d.field(1)
    d.apply(DWF_HDW, x, Ha, 1); d.apply(DWF_HDW, b2, Hb, 1)
    l, r_ = d.inner(x, Hb, 1)[0], d.inner(Ha, b2, 1)[0]
    assert abs(l - r_) / abs(l) < 1e-5
    del Ha, Hb, b2, psi
    # ---- 100 CG iterations on the even half: recursive residual == true residual, computed with
    # separately launched operator applications
    d.set_workspace(1, half_fields=5)                               # CG + Schur only: 5 x 12.2 GB
    hb = d.field_bytes(1, half=True) // 4
    b = x[:hb].clone()
    del x
    xs = d.field(1, half=True, zero=True)
    hist = np.array(d.cg_schur(b, xs, 100))
    assert np.all(np.diff(np.log(hist)) < 0.7) and hist[100] < hist[0]
    # true residual through the UNFUSED operator path (generic M_oo^-1 kernel, separate launches) on a second handle
    import os
    os.environ["DWF_NO_FUSE_MOOINV"] = "1"; os.environ["DWF_NO_FUSE_NORM"] = "1"
    try:
        d2 = Dwf(L4, LS4, M5, MASS4, DWF_F32)
    finally:
        del os.environ["DWF_NO_FUSE_MOOINV"], os.environ["DWF_NO_FUSE_NORM"]
    d2.set_gauge(U)
    del U
    d.set_workspace(1, half_fields=0)                               # hand the CG workspace back before the second handle takes its own
    d._ws = None
    d2.set_workspace(1, half_fields=1)
    w, q = d2.field(1, half=True), d2.field(1, half=True)
    l0 = d2.launch_count()
    d2.apply(DWF_SCHUR_EO, xs, w, 1)
    assert d2.launch_count() - l0 == 3                               # K1, M_oo^-1, K2: the unfused form
    d2.apply(DWF_SCHUR_EO | DWF_DAGGER, w, q, 1)
    rtrue = b - q
    r2 = d.norm2(rtrue, 1, half=True)[0]
    assert abs(r2 - hist[100]) / hist[100] < 1e-3, (r2, hist[100])
