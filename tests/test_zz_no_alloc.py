"""adock_local_search_noalloc (include/adock.h): the ADADELTA local search for callers that may not allocate device
memory.  Its chain state lives in a file-scope device array of the library (ADOCK_NOALLOC_SCRATCH_BYTES), shared by
every call and never cleared, so the checks are made on several calls in a row with different batch sizes:
  * against the existing path forced to the same kernel variant ('lane1': adock_local_search with a stream-ordered
    allocation): bit-equal genotypes, energies, iteration counts and per-iteration traces;
  * against the existing path as a caller gets it ('auto'): the energies E(x_0) of the trace at the plain energy
    tolerance of the parity tests, max(1e-4 |E|, 1e-3 kcal/mol), and the same iteration counts (later iterations of
    two fp32 summation orders part chaotically: tests/test_gpu_parity.py, ADADELTA section);
  * a batch beyond the array is rejected with ADOCK_ELIMIT and a message that names the sizes, and launches nothing; one just
    inside it runs.
Collected last (zz) and self-contained: it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

LSIT = 12


@pytest.fixture(scope="module")
def ctx(W):
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests")
    from paper_2007_03678_b200 import binding as B
    B.lib()
    B.adock_set_path("auto")
    grids, lig = W.make_config("drug")
    pd = dict(W.DEFAULT_PARAMS)
    pd.update(lsit=LSIT)
    gp = B.make_params(pd)
    gg = B.Grids.from_workload(grids)
    gl = B.Ligand.from_workload(gg, lig, gp)
    yield dict(B=B, grids=grids, lig=lig, gp=gp, gg=gg, gl=gl, dev=torch.device("cuda:0"))
    B.adock_set_path("auto")


def run(ctx, fn, G):
    """one local-search call on a copy of the starting genotypes G; returns host arrays"""
    dev, n = ctx["dev"], G.shape[0]
    d_g = torch.from_numpy(G).to(dev)
    d_E = torch.full((n,), -7.0, device=dev)
    d_it = torch.full((n,), -1, dtype=torch.int32, device=dev)
    d_tr = torch.full((n, LSIT), float("nan"), device=dev)
    fn(ctx["gg"], ctx["gl"], ctx["gp"], d_g, d_E, d_it, d_tr)
    torch.cuda.synchronize()
    return d_g.cpu().numpy(), d_E.cpu().numpy(), d_it.cpu().numpy(), d_tr.cpu().numpy()


def check_against_existing(ctx, W, n, seed):
    B = ctx["B"]
    G = W.make_genotypes(n, ctx["lig"].R, ctx["grids"], seed=seed, wall_tail=0.0)
    got = run(ctx, B.adock_local_search_noalloc, G)
    B.adock_set_path("lane1")                            # the existing path on the same kernel variant
    try:
        same = run(ctx, B.adock_local_search, G)
    finally:
        B.adock_set_path("auto")
    auto = run(ctx, B.adock_local_search, G)             # the existing path as a caller gets it
    for a, b, what in zip(got, same, ("genotypes", "energies", "iterations", "trace")):
        assert np.array_equal(a, b, equal_nan=True), f"n={n}: {what} differ from adock_local_search on the same kernel variant"
    E0, R0 = got[3][:, 0].astype(np.float64), auto[3][:, 0].astype(np.float64)
    assert np.isfinite(E0).all()
    assert (np.abs(E0 - R0) <= np.maximum(1e-4 * np.abs(R0), 1e-3)).all(), f"n={n}: E(x_0) off the existing path's"
    assert np.array_equal(got[2], auto[2]) and (got[2] == LSIT).all()
    assert (got[1] <= E0 + np.maximum(1e-4 * np.abs(E0), 1e-3)).all()        # best energy seen is never above the start's
    return got


def test_noalloc_local_search_matches_existing_path_on_calls_in_a_row(ctx, W):
    B = ctx["B"]
    B.adock_launch_count(True)                                       # returns the count so far and resets it
    first = check_against_existing(ctx, W, 1000, seed=71)           # ragged: 31 groups + 8 chains
    check_against_existing(ctx, W, 12000, seed=72)                  # overwrites the shared array with a larger batch ('auto' is a lane variant here)
    check_against_existing(ctx, W, 333, seed=73)                    # and a smaller one: stale columns beside the live ones
    again = check_against_existing(ctx, W, 1000, seed=71)           # the first batch once more: same results
    for a, b in zip(first, again):
        assert np.array_equal(a, b, equal_nan=True)
    assert B.adock_launch_count(False) == 12             # one kernel per call (4 x (noalloc + lane1 + auto))


def test_noalloc_local_search_rejects_a_batch_beyond_the_array(ctx, W):
    B, dev, R = ctx["B"], ctx["dev"], ctx["lig"].R
    n = 200_000                                                     # x (19 + 3R) x 4 bytes = 34 MB > 16 MiB
    d_g = torch.zeros((n, 7 + R), device=dev)
    d_g[:, 3] = 1.0
    d_E = torch.full((n,), -7.0, device=dev)
    before = B.adock_launch_count(False)
    with pytest.raises(B.AdockError) as ei:
        B.adock_local_search_noalloc(ctx["gg"], ctx["gl"], ctx["gp"], d_g, d_E)
    assert ei.value.code == -4                                      # ADOCK_ELIMIT
    assert "ADOCK_NOALLOC_SCRATCH_BYTES" in str(ei.value) and str(n) in str(ei.value)
    torch.cuda.synchronize()
    assert B.adock_launch_count(False) == before and (d_E.cpu().numpy() == -7.0).all()      # nothing ran
    # a batch just inside the limit still runs (the launch pads n to whole CTAs: at most 7 groups of 32 more)
    n_ok = (((16 << 20) // ((19 + 3 * R) * 4) - 8 * 32) // 32) * 32 - 5
    G = W.make_genotypes(n_ok, R, ctx["grids"], seed=74, wall_tail=0.0)
    g, E, it, tr = run(ctx, B.adock_local_search_noalloc, G)
    assert (it == LSIT).all() and np.isfinite(E).all()
