"""GPU parity of df_chem_ann_source_mmlp (NEXT-1: one MLP per species) against the oracle: the 16-bit
tensor path, judged like the single network (2e-2 normwise per species; element-wise max(2e-2, 1.25 x the floor of
an exactly rounded fp16 chain), A12); sum_k (Y_k + dY_k) = 1 to 1e-6 on every cell."""
import numpy as np
import pytest

from tests import helpers, ideal16

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


@pytest.mark.parametrize("K,hidden,n,ld", [(19, [128, 64, 32], 1000, 1000), (9, [64, 64, 48], 131, 132),
                                           (19, [1600, 800, 400], 300, 300)])
def test_mmlp_source(B, K, hidden, n, ld):
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    seed = synth.config_seed(2)
    mech = synth.make_mechanism(K, seed)
    nets = synth.make_mmlp(K, hidden, 1, seed)
    cells = synth.cells_stratified(K, n, seed, ld=ld)
    gm, gn = B.Mech(mech), B.AnnMmlp(nets)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    om_g, dY_g = torch.zeros(K, ld, device="cuda"), torch.zeros(K, ld, device="cuda")
    ws = B.alloc_workspace_mmlp(gn, n, ld)
    B.df_chem_ann_source_mmlp(gn, gm, T, p, Y, omega=om_g, dY=dY_g, workspace=ws, n_cells=n)
    torch.cuda.synchronize()
    om_g, dY_g = om_g.cpu().numpy(), dY_g.cpu().numpy()
    s = (cells.Y[:, :n].astype(np.float64) + dY_g[:, :n]).sum(axis=0)
    assert np.abs(s - 1.0).max() <= 1e-6
    om_r, dY_r = oracle.Mmlp(nets).source(oracle.Mech(mech), cells.T, cells.p, cells.Y[:, :n])
    floor_om, floor_dY = ideal16.ideal_chain_source_mmlp(mech, nets, cells.T, cells.p, cells.Y[:, :n], "fp16")
    failures = []
    for name, got, ref, ideal in (("dY", dY_g[:, :n], dY_r[:, :n], floor_dY), ("omega", om_g[:, :n], om_r[:, :n], floor_om)):
        table = helpers.mixed_err_table(got, ref)
        bound, floor = helpers.bounds_16bit(ref, ideal, 2e-2)
        helpers.record(f"mmlp_{K}_{hidden[0]}", dict(quantity=name, dims=[K + 2] + hidden + [1], precision=1, n=n, cells_compared=n,
                                                    sum_to_one=float(np.abs(s - 1.0).max()), tol=2e-2, per_species=table,
                                                    ideal_fp16_chain=floor))
        for t in table:
            if t["mixed"] > bound[t["k"]] or t["normwise"] > 2e-2:
                failures.append(f"{name}[k={t['k']}]: mixed {t['mixed']:.3e} (bound {bound[t['k']]:.3e}) normwise {t['normwise']:.3e}")
    assert not failures, "; ".join(failures)
    assert (om_g[:, n:] == 0).all()


def test_mmlp_errors(B):
    from paper_2312_05800_b200 import synth
    nets = synth.make_mmlp(9, [64, 64, 32], 1, 3)
    gn = B.AnnMmlp(nets)
    gm19 = B.Mech(synth.make_mechanism(19, 3))
    x = torch.zeros(64, device="cuda")
    with pytest.raises(B.DfError) as e:
        B.df_chem_ann_source_mmlp(gn, gm19, x, x, torch.zeros(19, 64, device="cuda"), omega=torch.zeros(19, 64, device="cuda"),
                                  workspace=torch.zeros(1 << 20, dtype=torch.uint8, device="cuda"))
    assert e.value.code == B.DF_ERR_INVALID_ARG
    nets[3].W[1][0, 0] = np.float32(0.1)     # not bf16-valued: refused like the single network
    with pytest.raises(B.DfError):
        B.AnnMmlp(nets)


def test_mmlp_source_bench_size(B):
    """NEXT-1 at the size bench.py times it (262,144 cells, 19 networks 21-1600-800-400-1): kernels on the whole field, oracle and
    fp16-chain floor on sampled cells (plus the end of the field), sum-to-one on every cell."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    K, hidden, n = 19, [1600, 800, 400], 262144
    seed = synth.config_seed(2)
    mech = synth.make_mechanism(K, seed)
    nets = synth.make_mmlp(K, hidden, 1, seed)
    cells = synth.cells_stratified(K, n, seed)
    gm, gn = B.Mech(mech), B.AnnMmlp(nets)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    om_g, dY_g = torch.zeros(K, n, device="cuda"), torch.zeros(K, n, device="cuda")
    ws = B.alloc_workspace_mmlp(gn, n, n)
    B.df_chem_ann_source_mmlp(gn, gm, T, p, Y, omega=om_g, dY=dY_g, workspace=ws, n_cells=n)
    torch.cuda.synchronize()
    s = (Y.double() + dY_g.double()).sum(dim=0)
    sum_err = float((s - 1.0).abs().max())
    assert sum_err <= 1e-6
    idx = np.unique(np.concatenate([np.arange(0, n, n // 160), np.arange(n - 40, n)]))
    it = torch.from_numpy(idx).cuda()
    Ys = np.ascontiguousarray(cells.Y[:, idx])
    om_r, dY_r = oracle.Mmlp(nets).source(oracle.Mech(mech), cells.T[idx], cells.p[idx], Ys)
    floor_om, floor_dY = ideal16.ideal_chain_source_mmlp(mech, nets, cells.T[idx], cells.p[idx], Ys, "fp16")
    failures = []
    for name, got, ref, ideal in (("dY", dY_g[:, it].cpu().numpy(), dY_r[:, :len(idx)], floor_dY),
                                  ("omega", om_g[:, it].cpu().numpy(), om_r[:, :len(idx)], floor_om)):
        table = helpers.mixed_err_table(got, ref)
        bound, floor = helpers.bounds_16bit(ref, ideal, 2e-2)
        helpers.record("mmlp_bench_size", dict(quantity=name, dims=[K + 2] + hidden + [1], precision=1, n=n, cells_compared=int(len(idx)),
                                               sum_to_one=sum_err, tol=2e-2, per_species=table, ideal_fp16_chain=floor))
        for t in table:
            if t["mixed"] > bound[t["k"]] or t["normwise"] > 2e-2:
                failures.append(f"{name}[k={t['k']}]: mixed {t['mixed']:.3e} (bound {bound[t['k']]:.3e}) normwise {t['normwise']:.3e}")
    assert not failures, "; ".join(failures)
