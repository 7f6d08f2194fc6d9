"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the kernels run on the whole
field, the oracle on a strided sample of cells (plus the whole ragged tail), and size-independent properties
(sum-to-one, positivity, convergence counter) are checked on every cell."""
import numpy as np
import pytest

from tests import helpers

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_05800_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def sample_idx(n, m=4096):
    return np.unique(np.concatenate([np.arange(0, n, max(1, n // m)), np.arange(max(0, n - 300), n)]))


def test_cfg3_full_pipeline(B):
    """configs[2]: 2,097,152 cells, K = 19, T_from_h -> properties -> 16-bit tensor MLP, as bench.py runs it."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    n, K = 2097152, 19
    mech, ann, cells = synth.make_config(3)
    om, oa = oracle.Mech(mech), oracle.Ann(ann)
    gm, ga = B.Mech(mech), B.Ann(ann)
    T0, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    h = torch.empty(n, device="cuda")
    B.df_thermo_properties(gm, T0, p, Y, h=h)              # the enthalpy field a solver would hold
    T = dev(cells.T_guess)
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    mu, lam = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    D, omega, dY = (torch.empty(K, n, device="cuda") for _ in range(3))
    B.df_thermo_T_from_h(gm, h, Y, T, n_unconverged=cnt)
    B.df_thermo_properties(gm, T, p, Y, mu=mu, lam=lam, D=D)
    B.df_chem_ann_source(ga, gm, T, p, Y, omega=omega, dY=dY, workspace=B.alloc_workspace(ga, n))
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0
    # properties that hold at any size, every cell
    s = (Y.double() + dY.double()).sum(dim=0)
    sum_err = float((s - 1.0).abs().max())
    assert sum_err <= 1e-6, sum_err
    assert bool((D > 0).all()) and bool((mu > 0).all()) and bool((lam > 0).all())
    # sampled cells against the oracle (A20: properties / ANN judged at the fp32 T the Newton call wrote)
    idx = sample_idx(n)
    hs, Ys, Ts = h.cpu().numpy()[idx], np.ascontiguousarray(cells.Y[:, idx]), T.cpu().numpy()[idx]
    T_ref = om.T_from_h(hs, Ys, cells.T_guess[idx])
    assert np.abs(Ts - T_ref).max() <= 1e-3
    ref = om.properties(Ts, cells.p[idx], Ys)
    for name, got in (("mu", mu), ("lam", lam)):
        assert helpers.rel_err(got.cpu().numpy()[idx], ref[name]).max() <= 1e-5, name
    assert helpers.rel_err(D.cpu().numpy()[:, idx], ref["D"][:, :len(idx)]).max() <= 1e-5
    om_r, dY_r = oa.source(om, Ts, cells.p[idx], Ys)
    from tests import ideal16
    ideal = dict(zip(("omega", "dY"), ideal16.ideal_chain_source(mech, ann, Ts, cells.p[idx], Ys, "fp16")))
    failures = []
    for name, got, r in (("dY", dY, dY_r), ("omega", omega, om_r)):
        r = r[:, :len(idx)]
        table = helpers.mixed_err_table(got.cpu().numpy()[:, idx], r)
        bound, floor = helpers.bounds_16bit(r, ideal[name], 2e-2)   # A12, 16-bit path: north_star's 2e-2
        helpers.record("cfg3_full_pipeline", dict(quantity=name, dims=list(ann.dims), precision=1, n=n, cells_compared=int(len(idx)),
                                                  sum_to_one=sum_err, tol=2e-2, per_species=table, ideal_fp16_chain=floor))
        for t in table:
            if t["mixed"] > bound[t["k"]] or t["normwise"] > 2e-2:
                failures.append(f"{name}[k={t['k']}]: mixed {t['mixed']:.3e} (bound {bound[t['k']]:.3e}) normwise {t['normwise']:.3e}")
    assert not failures, "; ".join(failures)


def test_cfg4_properties_K53(B):
    """configs[3]: 2,097,152 cells, K = 53, property pass only."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech, _, cells = synth.make_config(4)
    n, K = cells.n, 53
    gm = B.Mech(mech)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    out = {k: torch.empty(n, device="cuda") for k in ("cp", "h", "mu", "lam")}
    D = torch.empty(K, n, device="cuda")
    B.df_thermo_properties(gm, T, p, Y, D=D, **out)
    torch.cuda.synchronize()
    assert bool((D > 0).all()) and bool(torch.isfinite(D).all())
    idx = sample_idx(n, 2048)
    ref = oracle.Mech(mech).properties(cells.T[idx], cells.p[idx], np.ascontiguousarray(cells.Y[:, idx]))
    for k in ("cp", "mu", "lam"):
        assert helpers.rel_err(out[k].cpu().numpy()[idx], ref[k]).max() <= 1e-5, k
    eh = np.abs(out["h"].cpu().numpy()[idx] - ref["h"]) / np.maximum(np.abs(ref["h"]), ref["cp"] * cells.T[idx])
    assert eh.max() <= 1e-5
    assert helpers.rel_err(D.cpu().numpy()[:, idx], ref["D"][:, :len(idx)]).max() <= 1e-5


@pytest.mark.parametrize("guess", ["warm", "cold"])
def test_cfg5_T_from_h_robustness(B, guess):
    """configs[4]: 16,777,216 cells, K = 19, T in 250..3500 K, near-pure and 1e-20-trace cells."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech, _, cells = synth.make_config(5)
    n = cells.n
    gm = B.Mech(mech)
    Y = dev(cells.Y)
    h = torch.empty(n, device="cuda")
    B.df_thermo_properties(gm, dev(cells.T), None, Y, h=h)
    g = cells.T_guess if guess == "warm" else np.full(n, 1000.0, np.float32)
    T, cp = dev(g), torch.empty(n, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.df_thermo_T_from_h(gm, h, Y, T, cp=cp, n_unconverged=cnt)
    torch.cuda.synchronize()
    assert int(cnt.item()) == 0
    # the state was drawn at cells.T: the root must come back to it (fp32 h rounding moves it by < 1e-2 K)
    assert float((T - dev(cells.T)).abs().max()) <= 2e-2
    idx = sample_idx(n)
    om = oracle.Mech(mech)
    Ys = np.ascontiguousarray(cells.Y[:, idx])
    T_ref = om.T_from_h(h.cpu().numpy()[idx], Ys, g[idx])
    assert np.abs(T.cpu().numpy()[idx] - T_ref).max() <= 1e-3
    cp_ref, _ = om.mixture_cp_h(T.cpu().numpy()[idx], Ys)
    assert helpers.rel_err(cp.cpu().numpy()[idx], cp_ref).max() <= 1e-5


def test_full_size_extras_and_pasr(B):
    """NEXT-4 / NEXT-3 at the size bench.py times them (2,097,152 cells, K = 19): kernels on the whole field, the oracle on
    sampled cells; kappa in [0, 1) and the gate on every cell."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech, _, cells = synth.make_config(3)
    n, K = cells.n, mech.K
    om, gm = oracle.Mech(mech), B.Mech(mech)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    cp, lam = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    D = torch.empty(K, n, device="cuda")
    B.df_thermo_properties(gm, T, p, Y, cp=cp, lam=lam, D=D)
    rho, psi, alpha, s = (torch.empty(n, device="cuda") for _ in range(4))
    rhoD, hk = torch.empty(K, n, device="cuda"), torch.empty(K, n, device="cuda")
    B.df_thermo_extras(gm, T, p, Y, cp=cp, lam=lam, D=D, rho=rho, psi=psi, alpha=alpha, rhoD=rhoD, hk=hk, s=s)
    idx = sample_idx(n)
    it = torch.from_numpy(idx).cuda()
    pick = lambda t: t[..., it].cpu().numpy()
    ref = om.extras(cells.T[idx], cells.p[idx], np.ascontiguousarray(cells.Y[:, idx]), cp=pick(cp), lam=pick(lam), D=pick(D))
    for name, got in (("rho", rho), ("psi", psi), ("alpha", alpha), ("s", s)):
        e = helpers.rel_err(pick(got), ref[name])
        assert e.max() <= 1e-5, f"{name}: {e.max():.3e}"
    assert helpers.rel_err(pick(rhoD), ref["rhoD"][:, :len(idx)]).max() <= 1e-5
    scale = np.maximum(np.abs(ref["hk"][:, :len(idx)]), 3.5 * helpers.R * cells.T[idx][None, :].astype(np.float64) / mech.W[:, None])
    assert (np.abs(pick(hk) - ref["hk"][:, :len(idx)]) / scale).max() <= 1e-5
    assert bool((rho > 0).all()) and bool(torch.isfinite(s).all())

    g = torch.Generator(device="cuda").manual_seed(11)
    mu = torch.rand(n, device="cuda", generator=g) * 7e-5 + 1e-5
    ks = torch.rand(n, device="cuda", generator=g) * 10 + 0.01
    eps = torch.rand(n, device="cuda", generator=g) * 1e4 + 0.1
    omega = torch.randn(K, n, device="cuda", generator=g) * 50
    omega[:, :7] = 0.0
    om_in = pick(omega)
    kappa = torch.full((n,), -7.0, device="cuda")
    B.df_chem_pasr_scale(gm, T, p, Y, mu, ks, eps, 500.0, omega, kappa=kappa)
    torch.cuda.synchronize()
    oref, kref = om.pasr(cells.T[idx], cells.p[idx], np.ascontiguousarray(cells.Y[:, idx]), pick(mu), pick(ks), pick(eps), 500.0, om_in)
    assert np.abs(pick(kappa) - kref).max() <= 1e-5
    mixed, norm = helpers.mixed_err(pick(omega), oref[:, :len(idx)])
    assert mixed <= 1e-5 and norm <= 1e-5, (mixed, norm)
    assert bool(((kappa >= 0) & (kappa < 1)).all())
    assert bool((kappa[T < 500.0] == 0).all()) and bool((kappa[:7] == 0).all())
