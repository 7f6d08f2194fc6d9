"""GPU parity: every hot call through the C ABI vs the fp64 oracle, element by element, on the
same seeded fp32 inputs (SURVEY 8(c) "same input bits"; tolerances = DESIGN.md A12)."""
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


def h_from_T(omech, cells):
    """fp32 enthalpy field the way a solver would hold it: oracle h(T, Y) rounded once to fp32."""
    _, h = omech.mixture_cp_h(cells.T, cells.Y[:, :cells.n])
    return h.astype(np.float32)


def make_case(cfg, n, ld=None):
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech, ann, cells = synth.make_config(cfg, n=n, ld=ld)
    return mech, ann, cells, oracle.Mech(mech)


# --------------------------------------------------------------------------------------------
# H1: T from h
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n,ld", [(1, 4096, None), (5, 20003, 20004), (3, 8190, 8192), (4, 3001, 3004)])
@pytest.mark.parametrize("guess", ["warm", "cold", "invalid"])
def test_T_from_h(B, cfg, n, ld, guess):
    mech, _, cells, om = make_case(cfg, n, ld)
    h32 = h_from_T(om, cells)
    if guess == "warm":
        g = cells.T_guess.copy()
    elif guess == "cold":
        g = np.full(n, 1000.0, np.float32)
    else:
        g = np.zeros(n, np.float32)
        g[::3] = np.nan
        g[1::3] = -5.0
    T_ref = om.T_from_h(h32, cells.Y[:, :n], np.where(np.isfinite(g) & (g > 0), g, 1000.0))
    gm = B.Mech(mech)
    T = dev(g)
    cp = torch.empty_like(T)
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.df_thermo_T_from_h(gm, dev(h32), dev(cells.Y), T, cp=cp, n_unconverged=cnt)
    torch.cuda.synchronize()
    err = np.abs(T.cpu().numpy().astype(np.float64) - T_ref)
    assert err.max() <= 1e-3, f"max |dT| = {err.max():.3e} K at {err.argmax()}"
    assert int(cnt.item()) == 0
    cp_ref, _ = om.mixture_cp_h(T.cpu().numpy(), cells.Y[:, :n])
    assert helpers.rel_err(cp.cpu().numpy(), cp_ref).max() <= 1e-5


@pytest.mark.parametrize("n,ld", [(1, 4), (127, 128), (129, 132), (257, 260), (1000, 1000)])
@pytest.mark.parametrize("side", ["lo", "hi", "mid", "mixed"])
def test_T_from_h_range_sorted_blocks(B, n, ld, side):
    """The fixed-K kernel decides the NASA range of a cell before it iterates (hi iff h >= h(T_mid, Y)) and gives
    low-range cells an fp32 correction on top of the fp64 high-range coefficients: fields that are all lo, all hi, sit on
    T_mid (either polynomial is right there, A2) or mix both, at sizes around the warp / block boundaries (the ragged
    last block is a launch of its own), must all come back to the oracle's root; the pad between n and ld must stay
    untouched."""
    mech, _, cells, om = make_case(3, n, ld)
    rng = np.random.default_rng(n * 7 + len(side))
    if side == "lo":
        cells.T[:] = rng.uniform(300.0, 999.0, n)
    elif side == "hi":
        cells.T[:] = rng.uniform(1001.0, 3400.0, n)
    elif side == "mid":
        cells.T[:] = 1000.0 + rng.choice([0.0, 1e-3, -1e-3, 0.5, -0.5], n)
    h32 = h_from_T(om, cells)
    g = np.full(n, 1000.0, np.float32) if side == "mid" else rng.uniform(300.0, 3400.0, n).astype(np.float32)
    T_ref = om.T_from_h(h32, cells.Y[:, :n], g)
    gm = B.Mech(mech)
    Tbuf = torch.full((ld,), -7.0, device="cuda")
    Tbuf[:n] = dev(g)
    cp = torch.full((ld,), -7.0, device="cuda")
    hbuf = torch.zeros(ld, device="cuda")
    hbuf[:n] = dev(h32)
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.df_thermo_T_from_h(gm, hbuf, dev(cells.Y), Tbuf, cp=cp, n_unconverged=cnt, n_cells=n)
    torch.cuda.synchronize()
    Tg = Tbuf.cpu().numpy()
    assert np.abs(Tg[:n].astype(np.float64) - T_ref).max() <= 1e-3
    assert int(cnt.item()) == 0
    assert (Tg[n:] == -7.0).all() and (cp.cpu().numpy()[n:] == -7.0).all()
    cp_ref, _ = om.mixture_cp_h(Tg[:n], cells.Y[:, :n])
    assert helpers.rel_err(cp.cpu().numpy()[:n], cp_ref).max() <= 1e-5


def test_T_from_h_nan_cells_do_not_spread(B):
    """A18: NaN in h or Y must neither hang nor fault, is counted as unconverged, and leaves the other cells of the
    block (which share threads and shared-memory slots with it after the range sort) at the oracle's root."""
    n = 1500
    mech, _, cells, om = make_case(3, n)
    h32 = h_from_T(om, cells)
    Y = cells.Y.copy()
    bad = np.zeros(n, bool)
    bad[[0, 1, 130, 255, 256, 700, 1499]] = True
    h32[[0, 130, 256, 1499]] = np.nan
    Y[3, [1, 255, 700]] = np.nan
    T_ref = om.T_from_h(h32[~bad], np.ascontiguousarray(cells.Y[:, ~bad]), cells.T_guess[~bad])
    gm = B.Mech(mech)
    T = dev(cells.T_guess)
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.df_thermo_T_from_h(gm, dev(h32), dev(Y), T, n_unconverged=cnt)
    torch.cuda.synchronize()
    assert np.abs(T.cpu().numpy()[~bad].astype(np.float64) - T_ref).max() <= 1e-3
    assert int(cnt.item()) == int(bad.sum())


def test_T_from_h_empty_and_errors(B):
    mech, _, cells, om = make_case(1, 64)
    gm = B.Mech(mech)
    Y = dev(cells.Y)
    T = dev(cells.T_guess)
    h = dev(h_from_T(om, cells))
    B.df_thermo_T_from_h(gm, h, Y, T, n_cells=0)  # no-op
    with pytest.raises(B.DfError) as e:
        B.df_thermo_T_from_h(gm, h, Y, T, n_cells=65)  # ld < n
    assert e.value.code == B.DF_ERR_INVALID_ARG
    with pytest.raises(B.DfError):
        B.df_thermo_T_from_h(gm, h[1:], Y, T[1:], n_cells=60)  # misaligned


# --------------------------------------------------------------------------------------------
# H2: properties
# --------------------------------------------------------------------------------------------
def check_properties(B, mech, cells, om, n):
    gm = B.Mech(mech)
    K, ld = cells.Y.shape
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    out = {k: torch.empty(n, device="cuda") for k in ("cp", "h", "mu", "lam")}
    D = torch.zeros(K, ld, device="cuda")
    B.df_thermo_properties(gm, T, p, Y, D=D, **out)
    torch.cuda.synchronize()
    ref = om.properties(cells.T, cells.p, cells.Y[:, :n])
    for k in ("cp", "mu", "lam"):
        e = helpers.rel_err(out[k].cpu().numpy(), ref[k])
        assert e.max() <= 1e-5, f"{k}: max rel err {e.max():.3e} at {e.argmax()}"
    eh = np.abs(out["h"].cpu().numpy().astype(np.float64) - ref["h"]) / np.maximum(np.abs(ref["h"]), ref["cp"] * cells.T)
    assert eh.max() <= 1e-5, f"h: {eh.max():.3e}"
    eD = helpers.rel_err(D.cpu().numpy()[:, :n], ref["D"][:, :n])
    assert eD.max() <= 1e-5, f"D: max rel err {eD.max():.3e} at {np.unravel_index(eD.argmax(), eD.shape)}"


@pytest.mark.parametrize("cfg,n,ld", [(1, 4096, None), (3, 8190, 8192), (5, 20003, 20004), (4, 3001, 3004)])
def test_properties(B, cfg, n, ld):
    mech, _, cells, om = make_case(cfg, n, ld)
    check_properties(B, mech, cells, om, n)


@pytest.mark.parametrize("K", [1, 2, 3, 9, 19, 24, 53])
def test_properties_one_hot_and_generic_K(B, K):
    """Degenerate cells: pure species (A7 self-diffusion branch) and exact zeros, any K."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(K, 77 + K)
    n = 4 * K + 8
    Y = np.zeros((K, n), np.float32)
    for i in range(n):
        Y[i % K, i] = 1.0
    if K > 1:
        Y[:, -4:] = 0.0
        Y[0, -4:] = 0.25
        Y[K - 1, -4:] = 0.75
    rng = np.random.default_rng(K)
    cells = synth.Cells(n, rng.uniform(300, 3000, n).astype(np.float32), np.full(n, 2.0e5, np.float32), Y,
                        np.zeros(n, np.float32))
    check_properties(B, mech, cells, oracle.Mech(mech), n)


def test_properties_subset_outputs(B):
    mech, _, cells, om = make_case(1, 512)
    gm = B.Mech(mech)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    cp = torch.empty(512, device="cuda")
    B.df_thermo_properties(gm, T, p, Y, cp=cp)
    mu = torch.empty(512, device="cuda")
    B.df_thermo_properties(gm, T, None, Y, mu=mu)
    torch.cuda.synchronize()
    ref = om.properties(cells.T, cells.p, cells.Y)
    assert helpers.rel_err(cp.cpu().numpy(), ref["cp"]).max() <= 1e-5
    assert helpers.rel_err(mu.cpu().numpy(), ref["mu"]).max() <= 1e-5


@pytest.mark.parametrize("K,w_hi", [(40, 20.0), (40, 250.0), (61, 1200.0), (19, 20.0), (19, 44.0), (19, 400.0)])
def test_properties_factored_wilke_weight_ranges(B, K, w_hi):
    """The property kernels hold Wilke's B factored (any K: 8 or 12 terms; K = 19: 7 or 8 terms; chosen at create from the
    molecular weights) or, when the weights span too wide a range, in full: log-spaced weights 1 ... w_hi exercise the three
    cases of each kernel."""
    import dataclasses
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(K, 900 + K)
    mech = dataclasses.replace(mech, W=np.exp(np.linspace(0.0, np.log(w_hi), K)))
    cells = synth.cells_stratified(K, 333, 901 + K, ld=336)
    check_properties(B, mech, cells, oracle.Mech(mech), 333)


@pytest.mark.parametrize("K,n,ld", [(24, 200, 200), (53, 131, 132)])
def test_properties_subset_outputs_generic_K(B, K, n, ld):
    """The any-K kernel's instantiations for calls that want only some outputs, on full groups and a ragged last one."""
    from oracle import oracle
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(K, 500 + K)
    cells = synth.cells_stratified(K, n, 600 + K, ld=ld)
    om = oracle.Mech(mech)
    gm = B.Mech(mech)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    ref = om.properties(cells.T, cells.p, cells.Y[:, :n])
    for names in (("cp",), ("mu",), ("D",), ("h", "lam"), ("cp", "h", "mu", "lam")):
        out = {k: (torch.full((K, ld), -1.0, device="cuda") if k == "D" else torch.full((ld,), -1.0, device="cuda")) for k in names}
        B.df_thermo_properties(gm, T, p, Y, n_cells=n, **out)
        torch.cuda.synchronize()
        for k, v in out.items():
            g = v.cpu().numpy()
            if k == "D":
                assert helpers.rel_err(g[:, :n], ref["D"]).max() <= 1e-5, (names, k)
                assert (g[:, n:] == -1.0).all()
            elif k == "h":
                scale = np.maximum(np.abs(ref["h"]), ref["cp"] * cells.T[:n])
                assert (np.abs(g[:n] - ref["h"]) / scale).max() <= 1e-5, (names, k)
            else:
                assert helpers.rel_err(g[:n], ref[k]).max() <= 1e-5, (names, k)
            if k != "D":
                assert (g[n:] == -1.0).all()


# --------------------------------------------------------------------------------------------
# H3: ANN source, fp32 path
# --------------------------------------------------------------------------------------------
def check_source(B, mech, ann, cells, n, tol, sample=None, tag=None):
    """tol bounds both A12 forms per species: the element-wise mixed error and the normwise error.  The measured
    figures are recorded (gpurun_out/parity_measured.jsonl) whether the test passes or not."""
    from oracle import oracle
    gm, ga = B.Mech(mech), B.Ann(ann)
    K, ld = cells.Y.shape
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    om_g = torch.zeros(K, ld, device="cuda")
    dY_g = torch.zeros(K, ld, device="cuda")
    ws = B.alloc_workspace(ga, n)
    B.df_chem_ann_source(ga, gm, T, p, Y, omega=om_g, dY=dY_g, workspace=ws, n_cells=n)
    torch.cuda.synchronize()
    om_g, dY_g = om_g.cpu().numpy(), dY_g.cpu().numpy()
    # sum_k (Y_k + dY_k) = 1 on every cell (A11 / P:86)
    s = (cells.Y[:, :n].astype(np.float64) + dY_g[:, :n]).sum(axis=0)
    sum_err = float(np.abs(s - 1.0).max())
    idx = np.arange(n) if sample is None else sample
    o_mech, o_ann = oracle.Mech(mech), oracle.Ann(ann)
    om_r, dY_r = o_ann.source(o_mech, cells.T[idx], cells.p[idx], np.ascontiguousarray(cells.Y[:, idx]))
    ideal = None
    if ann.precision == 1:   # the floor an exactly rounded fp16 chain has on these cells (tests/ideal16.py, A12)
        from tests import ideal16
        ideal = dict(zip(("omega", "dY"), ideal16.ideal_chain_source(mech, ann, cells.T[idx], cells.p[idx],
                                                                      np.ascontiguousarray(cells.Y[:, idx]), "fp16")))
    failures = []
    for name, got, ref in (("dY", dY_g[:, idx], dY_r), ("omega", om_g[:, idx], om_r)):
        ref = ref[:, :len(idx)]
        table = helpers.mixed_err_table(got, ref)
        bound, floor = (np.full(K, tol), None) if ideal is None else helpers.bounds_16bit(ref, ideal[name], tol)
        helpers.record(tag or "check_source", dict(quantity=name, dims=list(ann.dims), precision=int(ann.precision), n=int(n),
                                                   cells_compared=int(len(idx)), sum_to_one=sum_err, tol=tol,
                                                   per_species=table, ideal_fp16_chain=floor))
        for t in table:
            if t["mixed"] > bound[t["k"]] or t["normwise"] > tol:
                failures.append(f"{name}[k={t['k']}]: mixed {t['mixed']:.3e} (bound {bound[t['k']]:.3e}) normwise "
                                f"{t['normwise']:.3e} (bound {tol})")
    assert sum_err <= 1e-6, sum_err
    assert not failures, "; ".join(failures)
    return dY_g, om_g


def test_ann_source_fp32_cfg1(B):
    mech, ann, cells, _ = make_case(1, 4096)
    check_source(B, mech, ann, cells, 4096, 1e-5, tag="fp32_cfg1")


def test_ann_source_fp32_ragged_and_degenerate(B):
    from paper_2312_05800_b200 import synth
    mech, ann, cells, _ = make_case(1, 1003, 1004)
    cells.Y[:, :8] = 0.0
    cells.Y[np.arange(8), np.arange(8)] = 1.0   # one-hot cells: Y_k = 0 branch of the inverse transform
    check_source(B, mech, ann, cells, 1003, 1e-5, tag="fp32_ragged_degenerate")


@pytest.mark.parametrize("hidden", [[256, 200], [40], [24, 24, 24, 24, 24]])
def test_ann_source_fp32_other_shapes(B, hidden):
    """The fp32 path stages a layer's weights in shared memory when every layer fits (16 K floats); [256, 200] does not and
    reads them from global memory; one hidden layer and five hidden layers exercise the double buffering."""
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(9, 41)
    ann = synth.make_ann(9, hidden, 0, 42)
    cells = synth.cells_dirichlet(9, 333, 43, ld=336)
    check_source(B, mech, ann, cells, 333, 1e-5, tag="fp32_shapes_" + "_".join(map(str, hidden)))


def test_ann_K_mismatch(B):
    from paper_2312_05800_b200 import synth
    mech9 = B.Mech(synth.make_mechanism(9, 1))
    ann19 = B.Ann(synth.make_ann(19, [32, 32], 0, 1))
    x = torch.zeros(64, device="cuda")
    with pytest.raises(B.DfError) as e:
        B.df_chem_ann_source(ann19, mech9, x, x, torch.zeros(19, 64, device="cuda"), omega=torch.zeros(19, 64, device="cuda"))
    assert e.value.code == B.DF_ERR_INVALID_ARG


# --------------------------------------------------------------------------------------------
# H3: ANN source, bf16 / tcgen05 path (tolerance 2e-2, A12)
# --------------------------------------------------------------------------------------------
# north_star: "2e-2 relative on the bf16 path"; A12 reads it per species both element-wise, as
# |d| <= 2e-2 (|ref| + RMS_cells(ref_k)), and normwise.  Both at 2e-2; the measured figures are recorded.
@pytest.mark.parametrize("hidden,n,ld", [([128, 64, 32], 1000, 1000), ([64, 64, 48], 131, 132), ([192, 96, 80], 700, 704)])
def test_ann_source_bf16_small_nets(B, hidden, n, ld):
    """Small layer widths exercise the chunk/piece bookkeeping of the chain at sizes the oracle does in full."""
    from paper_2312_05800_b200 import synth
    mech = synth.make_mechanism(19, synth.config_seed(2))
    ann = synth.make_ann(19, hidden, 1, synth.config_seed(2))
    cells = synth.cells_stratified(19, n, synth.config_seed(2), ld=ld)
    check_source(B, mech, ann, cells, n, 2e-2, tag=f"bf16_small_{hidden[0]}_{hidden[1]}_{hidden[2]}")


@pytest.mark.parametrize("n", [128, 2077])
def test_ann_source_bf16_paper_net(B, n):
    """21 -> 1600 -> 800 -> 400 -> 19, every cell against the oracle; 2077 = 16 tiles + ragged tail."""
    mech, ann, cells, _ = make_case(2, n, (n + 3) // 4 * 4)
    check_source(B, mech, ann, cells, n, 2e-2, tag=f"bf16_paper_net_n{n}")


def test_ann_source_bf16_multi_tile_per_cta(B):
    """More tiles than SMs (each CTA loops) on the paper's net: sampled cells vs oracle, sum-to-one on all."""
    n = 148 * 128 * 2 + 77
    mech, ann, cells, _ = make_case(2, n, (n + 3) // 4 * 4)
    sample = np.unique(np.concatenate([np.arange(0, n, 97), np.arange(n - 130, n)]))
    check_source(B, mech, ann, cells, n, 2e-2, sample=sample, tag="bf16_paper_net_multi_tile")


def test_ann_create_precision1_contract(B):
    """include/df_thermo.h: precision 1 takes bf16-valued weights inside the fp16 range (the tensor path holds them
    in fp16, A21); anything else is refused instead of being re-rounded silently."""
    from paper_2312_05800_b200 import synth
    ann = synth.make_ann(19, [64, 64, 32], 1, 5)
    B.Ann(ann)                                   # the generator's bf16-rounded weights are accepted
    ann.W[1][3, 5] = np.float32(7.0e4)           # bf16-valued, but above 65504
    with pytest.raises(B.DfError) as e:
        B.Ann(ann)
    assert e.value.code == B.DF_ERR_UNSUPPORTED
    ann.W[1][3, 5] = np.float32(0.1)             # 0.1 is not bf16-representable
    with pytest.raises(B.DfError) as e:
        B.Ann(ann)
    assert e.value.code == B.DF_ERR_INVALID_ARG
    ann.W[1][3, 5] = np.float32(0.125)
    ann.b[2][0] = np.float32(np.inf)
    with pytest.raises(B.DfError) as e:
        B.Ann(ann)
    assert e.value.code == B.DF_ERR_UNSUPPORTED


def test_ann_two_live_handles_of_different_shapes(B):
    """Creating a small net after a large one must not break launches of the large one (the dynamic shared-memory
    attribute of the kernel is per device and fixed, not per handle)."""
    from paper_2312_05800_b200 import synth
    seed = synth.config_seed(2)
    mech = synth.make_mechanism(19, seed)
    big, small = synth.make_ann(19, [1600, 800, 400], 1, seed), synth.make_ann(19, [64, 64, 32], 1, seed)
    cells = synth.cells_stratified(19, 300, seed)
    gm, gb = B.Mech(mech), B.Ann(big)
    gs = B.Ann(small)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    o1, o2, o3 = (torch.zeros(19, 300, device="cuda") for _ in range(3))
    B.df_chem_ann_source(gb, gm, T, p, Y, omega=o1, workspace=B.alloc_workspace(gb, 300))
    B.df_chem_ann_source(gs, gm, T, p, Y, omega=o2, workspace=B.alloc_workspace(gs, 300))
    B.df_chem_ann_source(gb, gm, T, p, Y, omega=o3, workspace=B.alloc_workspace(gb, 300))
    torch.cuda.synchronize()
    assert float((o1 - o3).abs().max()) <= 1e-3 * float(o1.abs().max())
    assert float(o2.abs().max()) > 0


# --------------------------------------------------------------------------------------------
# df_step_host: the whole path over HOST arrays, pipelined in slices (include/df_thermo.h)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n,ld", [(1, 4097, 4100), (1, 150001, 150004), (3, 140003, 140004)])
def test_step_host_matches_device_path_and_oracle(B, cfg, n, ld):
    """Several slices (n > 2 x 65536), a ragged last slice and ld > n: the host step must give what the three
    device calls give on the same inputs (same kernels: T, cp, mu, lambda, D bit for bit; omega bit for bit on the
    fp32 path, within the run-to-run bound of DESIGN.md on the 16-bit path), and T must match the oracle."""
    mech, ann, cells, om = make_case(cfg, n, ld)
    K = mech.K
    h32 = h_from_T(om, cells)
    gm, ga = B.Mech(mech), B.Ann(ann)
    # device path
    dY, dp = dev(cells.Y), dev(cells.p)
    T = dev(cells.T_guess.copy())
    B.df_thermo_T_from_h(gm, dev(h32), dY, T)
    cp, mu, lam = (torch.empty(n, device="cuda") for _ in range(3))
    D, omg = torch.zeros(K, ld, device="cuda"), torch.zeros(K, ld, device="cuda")
    B.df_thermo_properties(gm, T, dp, dY, cp=cp, mu=mu, lam=lam, D=D)
    B.df_chem_ann_source(ga, gm, T, dp, dY, omega=omg, workspace=B.alloc_workspace(ga, n))
    torch.cuda.synchronize()
    # host path
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    oT, ocp, omu, olam = (torch.zeros(n).pin_memory() for _ in range(4))
    oD, oom = torch.zeros(K, ld).pin_memory(), torch.zeros(K, ld).pin_memory()
    ctx = B.HostCtx(gm, ga, n)
    for _ in range(2):   # the second call reuses the staging buffers
        ctx.step(n, ld, pin(h32), pin(cells.p), pin(cells.T_guess), pin(cells.Y), T=oT, cp=ocp, mu=omu, lam=olam, D=oD,
                 omega=oom)
    ctx.close()
    assert np.array_equal(oT.numpy(), T.cpu().numpy())
    assert np.array_equal(ocp.numpy(), cp.cpu().numpy())
    assert np.array_equal(omu.numpy(), mu.cpu().numpy())
    assert np.array_equal(olam.numpy(), lam.cpu().numpy())
    assert np.array_equal(oD.numpy()[:, :n], D.cpu().numpy()[:, :n])
    a, b = oom.numpy()[:, :n].astype(np.float64), omg.cpu().numpy()[:, :n].astype(np.float64)
    if ann.precision == 0:
        assert np.array_equal(a, b)
    else:
        nw = np.linalg.norm(a - b, axis=1) / np.maximum(np.linalg.norm(b, axis=1), 1e-300)
        assert nw.max() <= 1e-3, nw.max()
    assert np.all(oom.numpy()[:, n:] == 0) and np.all(oD.numpy()[:, n:] == 0)   # pitch padding untouched
    T_ref = om.T_from_h(h32, cells.Y[:, :n], cells.T_guess)
    assert np.abs(oT.numpy() - T_ref).max() <= 1e-3


def test_ann_tensor_path_reuses_scratch_across_launches(B):
    """The 16-bit path hands H2 from its drain to its TMA loads through a per-CTA scratch: a launch on other data in
    between must not leak into the next one (differences stay at the accumulation-order level)."""
    from paper_2312_05800_b200 import synth
    mech, ann, cells, _ = make_case(3, 148 * 128 * 6 + 76)   # ragged last tile, ld % 4 == 0
    other = synth.cells_stratified(mech.K, cells.n, 12345)
    gm, ga = B.Mech(mech), B.Ann(ann)
    ws = B.alloc_workspace(ga, cells.n)
    a = [dev(x) for x in (cells.T, cells.p, cells.Y)]
    b = [dev(x) for x in (other.T, other.p, other.Y)]
    ref, out, tmp = (torch.empty(mech.K, cells.n, device="cuda") for _ in range(3))
    B.df_chem_ann_source(ga, gm, *a, omega=ref, workspace=ws)
    for _ in range(4):
        B.df_chem_ann_source(ga, gm, *b, omega=tmp, workspace=ws)
        B.df_chem_ann_source(ga, gm, *a, omega=out, workspace=ws)
        torch.cuda.synchronize()
        nw = ((out - ref).double().norm(dim=1) / ref.double().norm(dim=1)).max().item()
        assert nw <= 1e-3, nw


# --------------------------------------------------------------------------------------------
# df_step_plan / df_thermochem_step: the step as one CUDA graph launch (NEXT-2)
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n,ld", [(1, 4097, 4100), (3, 20001, 20004)])
def test_step_plan_matches_the_three_calls(B, cfg, n, ld):
    """Replaying the captured step (twice: the graph must be re-launchable) gives what the three calls give on the same
    arrays: bit for bit for T, cp, mu, lambda, D and the fp32-path omega; within the run-to-run bound on the 16-bit path."""
    mech, ann, cells, om = make_case(cfg, n, ld)
    K = mech.K
    h32 = h_from_T(om, cells)
    gm, ga = B.Mech(mech), B.Ann(ann)
    dh, dp, dY, dTg = dev(h32), dev(cells.p), dev(cells.Y), dev(cells.T_guess)
    ws = B.alloc_workspace(ga, n)
    # the three calls
    T = dTg.clone()
    B.df_thermo_T_from_h(gm, dh, dY, T)
    cp, mu, lam = (torch.empty(n, device="cuda") for _ in range(3))
    D, omg = torch.zeros(K, ld, device="cuda"), torch.zeros(K, ld, device="cuda")
    B.df_thermo_properties(gm, T, dp, dY, cp=cp, mu=mu, lam=lam, D=D)
    B.df_chem_ann_source(ga, gm, T, dp, dY, omega=omg, workspace=ws)
    torch.cuda.synchronize()
    # the plan
    T2 = torch.full((n,), -1.0, device="cuda")
    cp2, mu2, lam2 = (torch.empty(n, device="cuda") for _ in range(3))
    D2, om2 = torch.zeros(K, ld, device="cuda"), torch.zeros(K, ld, device="cuda")
    plan = B.StepPlan(gm, ga, dh, dp, dY, T2, T_guess=dTg, cp=cp2, mu=mu2, lam=lam2, D=D2, omega=om2, workspace=ws)
    for _ in range(2):
        plan.launch()
    torch.cuda.synchronize()
    for a, b in ((T, T2), (cp, cp2), (mu, mu2), (lam, lam2), (D, D2)):
        assert torch.equal(a, b)
    if ann.precision == 0:
        assert torch.equal(omg, om2)
    else:
        nw = ((omg - om2).double().norm(dim=1) / omg.double().norm(dim=1)).max().item()
        assert nw <= 1e-3, nw
    T_ref = om.T_from_h(h32, cells.Y[:, :n], cells.T_guess)
    assert np.abs(T2.cpu().numpy() - T_ref).max() <= 1e-3
    plan.close()
