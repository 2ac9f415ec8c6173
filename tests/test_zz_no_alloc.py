"""The no-allocation entry point (include/ffpp_noalloc.h): ffpp_heatmap_entropy_noalloc keeps its scratch in a static
256 KiB device array of the library instead of handle memory.  Checked against the existing path (ffpp_heatmap_stats'
out_entropy / out_degree) within the tolerance the f1 tests use (1e-9 absolute; the two share arithmetic and summation
order, so they are in fact equal), on two calls in a row with different inputs (the shared array keeps the first call's
contents), and against the oracle.  Collected last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env(oracle_mod, gen_mod):
    import torch
    import paper_2512_07009_b200 as m
    assert torch.cuda.is_available()
    m.load_library()
    return torch, m, oracle_mod, gen_mod


def _grids(oracle, gen, seed_offset, B):
    w = gen.make_config(2, B=B, seed_offset=seed_offset)                 # 640x640 frames -> 80x80 grids, cell 8 px
    ref = oracle.run(w.params, w.raw, w.N_per_frame, w.frame_dims)       # the ORACLE's density grids are the input
    return w, ref.density.reshape(B, 80, 80)


def test_noalloc_entropy_matches_the_existing_path_on_two_calls_in_a_row(env):
    torch, m, oracle, gen = env
    B = 6
    w, _ = _grids(oracle, gen, 0, B)
    pp = m.FFPP.for_workload(w)
    ent = torch.empty(B, dtype=torch.float64, device="cuda")
    deg = torch.empty(B, dtype=torch.float64, device="cuda")
    for call, seed_offset in enumerate((0, 5)):                          # second call: other inputs, same static scratch
        w, D = _grids(oracle, gen, seed_offset, B)
        if call == 1:
            D = D.copy()
            D[1] = 0.0                                                   # an empty grid: entropy 0, degree 0
            D[2] = 0.25                                                  # a uniform grid: entropy ln(6400), degree 0
        dens = torch.from_numpy(np.ascontiguousarray(D)).cuda()
        ent.fill_(-1.0); deg.fill_(-1.0)
        m.heatmap_entropy_noalloc(dens, 80, 80, ent, deg)
        old = pp.heatmap_stats(dens.reshape(-1), w.frame_dims, 0.05, connectivity=4, max_regions=64)    # the existing path
        torch.cuda.synchronize()
        e_new, d_new = ent.cpu().numpy(), deg.cpu().numpy()
        e_old, d_old = old["entropy"].cpu().numpy(), old["degree"].cpu().numpy()
        assert np.abs(e_new - e_old).max() <= 1e-9 and np.abs(d_new - d_old).max() <= 1e-9, (call, e_new, e_old)
        assert np.array_equal(e_new, e_old) and np.array_equal(d_new, d_old), "same arithmetic and order: bit-identical"
        for f in range(B):
            assert abs(e_new[f] - oracle.entropy(D[f])) <= 1e-9 and abs(d_new[f] - oracle.clustering_degree(D[f])) <= 1e-9
        if call == 1:
            assert e_new[1] == 0.0 and d_new[1] == 0.0
            assert abs(e_new[2] - np.log(6400.0)) <= 1e-9 and abs(d_new[2]) <= 1e-9


def test_noalloc_entropy_ragged_tail_and_the_stated_limit(env):
    """a grid size that is not a multiple of the 2048-cell block (one block and many blocks per grid); a batch beyond
    FFPP_NOALLOC_MAX_BLOCKS is refused with FFPP_ECAPACITY and a message that names the limit; B = 0 is a no-op."""
    torch, m, oracle, gen = env
    rng = np.random.default_rng(7)
    for B, gh, gw in [(3, 17, 23), (2, 136, 240), (1, 1, 1)]:
        D = rng.gamma(0.4, 1.0, (B, gh, gw)).astype(np.float32)
        D[rng.random(D.shape) < 0.4] = 0.0
        ent = torch.empty(B, dtype=torch.float64, device="cuda"); deg = torch.empty(B, dtype=torch.float64, device="cuda")
        for _ in range(2):
            m.heatmap_entropy_noalloc(torch.from_numpy(D).cuda(), gw, gh, ent, deg)
        torch.cuda.synchronize()
        for f in range(B):
            assert abs(float(ent[f]) - oracle.entropy(D[f])) <= 1e-9
            assert abs(float(deg[f]) - oracle.clustering_degree(D[f])) <= 1e-9
    # limit: 4 blocks per 80x80 grid -> 4097 grids need 16388 > 16384 blocks
    B = m.NOALLOC_MAX_BLOCKS // 4 + 1
    dens = torch.zeros((B, 80, 80), dtype=torch.float32, device="cuda")
    ent = torch.empty(B, dtype=torch.float64, device="cuda"); deg = torch.empty(B, dtype=torch.float64, device="cuda")
    with pytest.raises(m.FFPPError) as ei:
        m.heatmap_entropy_noalloc(dens, 80, 80, ent, deg)
    assert ei.value.code == m.FFPP_ECAPACITY and "16384" in str(ei.value)
    m.heatmap_entropy_noalloc(dens[:B - 1], 80, 80, ent[:B - 1], deg[:B - 1])        # exactly at the limit: accepted
    torch.cuda.synchronize()
    assert float(ent[:B - 1].abs().max()) == 0.0
    lib = m.load_library()
    assert lib.ffpp_heatmap_entropy_noalloc(None, 0, 80, 80, None, None, None) == m.FFPP_OK
