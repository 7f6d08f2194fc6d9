"""GPU parity of df_thermo_extras (NEXT-4, A22) and df_chem_pasr_scale (NEXT-3, A23) against the fp64 oracle on the
same fp32 input bits.  Tolerances (A12 extended): positive quantities 1e-5 relative; h_k:
|d| <= 1e-5 max(|h_k|, 3.5 R T / W_k); s: 1e-5 relative; kappa: 1e-5 absolute (it lives in [0, 1)); scaled omega:
1e-5 (|ref| + RMS_k) and exactly 0 where the oracle gates."""
import numpy as np
import pytest

from tests import helpers

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")
R = helpers.R


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_05800_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


@pytest.mark.parametrize("cfg,n,ld", [(1, 4096, None), (3, 8190, 8192), (5, 20003, 20004), (4, 3001, 3004)])
def test_extras(B, cfg, n, ld):
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech, _, cells = synth.make_config(cfg, n=n, ld=ld)
    K, ldy = cells.Y.shape
    om, gm = oracle.Mech(mech), B.Mech(mech)
    rng = np.random.default_rng(cfg)
    p = (cells.p * rng.uniform(0.5, 3.0, n)).astype(np.float32)
    T, pd, Y = dev(cells.T), dev(p), dev(cells.Y)
    cp, lam = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    D = torch.zeros(K, ldy, device="cuda")
    B.df_thermo_properties(gm, T, pd, Y, cp=cp, lam=lam, D=D)
    rho, psi, alpha, s = (torch.full((n,), -7.0, device="cuda") for _ in range(4))
    rhoD, hk = torch.full((K, ldy), -7.0, device="cuda"), torch.full((K, ldy), -7.0, device="cuda")
    B.df_thermo_extras(gm, T, pd, Y, cp=cp, lam=lam, D=D, rho=rho, psi=psi, alpha=alpha, rhoD=rhoD, hk=hk, s=s)
    torch.cuda.synchronize()
    ref = om.extras(cells.T, p, cells.Y[:, :n], cp=cp.cpu().numpy(), lam=lam.cpu().numpy(), D=D.cpu().numpy()[:, :n])
    for name, got in (("rho", rho), ("psi", psi), ("alpha", alpha), ("s", s)):
        e = helpers.rel_err(got.cpu().numpy(), ref[name])
        assert e.max() <= 1e-5, f"{name}: {e.max():.3e} at {e.argmax()}"
    e = helpers.rel_err(rhoD.cpu().numpy()[:, :n], ref["rhoD"][:, :n])
    assert e.max() <= 1e-5, f"rhoD: {e.max():.3e}"
    scale = np.maximum(np.abs(ref["hk"][:, :n]), 3.5 * R * cells.T[None, :].astype(np.float64) / mech.W[:, None])
    eh = np.abs(hk.cpu().numpy()[:, :n] - ref["hk"][:, :n]) / scale
    assert eh.max() <= 1e-5, f"hk: {eh.max():.3e}"
    assert (rhoD.cpu().numpy()[:, n:] == -7.0).all() and (hk.cpu().numpy()[:, n:] == -7.0).all()   # pitch padding untouched


def test_extras_subsets_one_hot_and_errors(B):
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(3, 11)
    n = 8
    Y = np.zeros((3, n), np.float32)
    Y[np.arange(n) % 3, np.arange(n)] = 1.0          # pure cells: X_k = 0 terms of the entropy drop out
    T = np.linspace(300, 3000, n).astype(np.float32)
    p = np.full(n, 2.0e5, np.float32)
    gm, om = B.Mech(mech), oracle.Mech(mech)
    s, rho = torch.empty(n, device="cuda"), torch.empty(n, device="cuda")
    B.df_thermo_extras(gm, dev(T), dev(p), dev(Y), s=s)
    B.df_thermo_extras(gm, dev(T), dev(p), dev(Y), rho=rho)
    torch.cuda.synchronize()
    ref = om.extras(T, p, Y)
    assert helpers.rel_err(s.cpu().numpy(), ref["s"]).max() <= 1e-5
    assert helpers.rel_err(rho.cpu().numpy(), ref["rho"]).max() <= 1e-5
    with pytest.raises(B.DfError) as e:
        B.df_thermo_extras(gm, dev(T), dev(p), dev(Y), alpha=rho)      # alpha needs cp and lambda
    assert e.value.code == B.DF_ERR_INVALID_ARG
    B.df_thermo_extras(gm, dev(T), dev(p), dev(Y), rho=rho, n_cells=0)  # no-op


@pytest.mark.parametrize("cfg,n,ld", [(1, 4099, 4100), (3, 8190, 8192), (4, 3001, 3004)])
def test_pasr_scale(B, cfg, n, ld):
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech, _, cells = synth.make_config(cfg, n=n, ld=ld)
    K, ldy = cells.Y.shape
    om, gm = oracle.Mech(mech), B.Mech(mech)
    rng = np.random.default_rng(100 + cfg)
    mu = rng.uniform(1e-5, 8e-5, n).astype(np.float32)
    ks = rng.uniform(0.01, 10.0, n).astype(np.float32)
    eps = rng.uniform(0.1, 1e4, n).astype(np.float32)
    omega = np.zeros((K, ldy), np.float32)
    omega[:, :n] = rng.normal(0.0, 50.0, (K, n))
    omega[:, :7] = 0.0                               # cells where nothing reacts
    omega[0, 7:40] = 0.0                             # a species that does not react in some cells
    g_om = dev(omega)
    kappa = torch.full((n,), -7.0, device="cuda")
    B.df_chem_pasr_scale(gm, dev(cells.T), dev(cells.p), dev(cells.Y), dev(mu), dev(ks), dev(eps), 500.0, g_om, kappa=kappa)
    torch.cuda.synchronize()
    ref, kref = om.pasr(cells.T, cells.p, cells.Y[:, :n], mu, ks, eps, 500.0, omega[:, :n])
    kg = kappa.cpu().numpy()
    assert np.abs(kg - kref).max() <= 1e-5
    assert (kg[kref == 0] == 0).all()                # the gate and the no-reaction cells exactly
    assert (cells.T < 500.0).any()
    mixed, norm = helpers.mixed_err(g_om.cpu().numpy()[:, :n], ref[:, :n])
    assert mixed <= 1e-5 and norm <= 1e-5, (mixed, norm)
    assert (g_om.cpu().numpy()[:, n:] == 0).all()
