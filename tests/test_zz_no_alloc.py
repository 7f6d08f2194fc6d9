"""df_chem_ann_source_static (include/df_thermo.h): the tensor-path ANN source on the library's static device scratch.

Outside SURVEY 8 on purpose: an entry point for callers that may not allocate.  It runs the same kernel as
df_chem_ann_source, so the test compares the two on the same inputs, with the A12 tolerance the 16-bit path's parity
tests use (2e-2, element-wise mixed and normwise; the two runs differ only by the issuer race of DESIGN.md 6, ~1e-4), on
two calls in a row with different fields and sizes -- the second call finds the first call's contents in the shared array.
The file sorts last so that, under `pytest -x`, a failure here cannot hide another test.

The size rejection (scratch need > DF_ANN_STATIC_SCRATCH_BYTES) cannot be provoked on a 148-SM device: the largest
network the tensor path accepts (d2 = 800) needs 29.4 MiB there.  The other rejection (fp32 handle) is tested.
"""
import numpy as np
import pytest

from tests import helpers

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = 2e-2   # A12, the 16-bit path


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2312_05800_b200 import binding
    return binding


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_static_scratch_matches_workspace_path_twice(B):
    from paper_2312_05800_b200 import synth
    mech, ann, cells_a = synth.make_config(3, n=37965, ld=37968)     # 297 tiles: full grid, 29.4 MiB of the scratch, ragged
    cells_b = synth.cells_stratified(mech.K, 2077, 4242, ld=2080)    # 17 tiles: a different field through the same array
    assert ann.precision == 1
    gm, ga = B.Mech(mech), B.Ann(ann)
    K = mech.K
    assert ga.workspace_bytes(37965) <= B.df_ann_static_scratch_bytes() == 32 << 20

    fields, ref, got = [], [], []
    for cells in (cells_a, cells_b):
        n, ld = cells.n, cells.Y.shape[1]
        T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
        fields.append((n, T, p, Y))
        om, dY = torch.zeros(K, ld, device="cuda"), torch.zeros(K, ld, device="cuda")
        B.df_chem_ann_source(ga, gm, T, p, Y, omega=om, dY=dY, workspace=B.alloc_workspace(ga, n), n_cells=n)   # existing path
        ref.append((om, dY))
        got.append((torch.full((K, ld), 7.0, device="cuda"), torch.full((K, ld), 7.0, device="cuda")))
    B.df_chem_ann_source_static(ga, gm, fields[0][1], fields[0][2], fields[0][3], n_cells=0)   # per-device set-up only
    torch.cuda.synchronize()

    free_before = torch.cuda.mem_get_info()[0]
    for (n, T, p, Y), (om, dY) in zip(fields, got):              # two calls in a row, same stream
        B.df_chem_ann_source_static(ga, gm, T, p, Y, omega=om, dY=dY, n_cells=n)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated or freed by the calls"

    for (n, _, _, _), (om_r, dY_r), (om_g, dY_g) in zip(fields, ref, got):
        assert bool((om_g[:, n:] == 7.0).all()) and bool((dY_g[:, n:] == 7.0).all())   # the pad is not written
        for name, g, r in (("omega", om_g, om_r), ("dY", dY_g, dY_r)):
            g, r = g[:, :n].cpu().numpy().astype(np.float64), r[:, :n].cpu().numpy().astype(np.float64)
            assert np.isfinite(g).all()
            for t in helpers.mixed_err_table(g, r):
                assert t["mixed"] <= TOL and t["normwise"] <= TOL, (name, n, t)


def test_static_scratch_rejects_fp32_handle(B):
    from paper_2312_05800_b200 import synth
    mech, ann, cells = synth.make_config(1, n=256)
    assert ann.precision == 0
    gm, ga = B.Mech(mech), B.Ann(ann)
    T, p, Y = dev(cells.T), dev(cells.p), dev(cells.Y)
    om = torch.zeros(mech.K, cells.Y.shape[1], device="cuda")
    with pytest.raises(B.DfError) as e:
        B.df_chem_ann_source_static(ga, gm, T, p, Y, omega=om, n_cells=256)
    assert e.value.code == B.DF_ERR_UNSUPPORTED
