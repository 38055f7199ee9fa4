"""-m gpu: the widened rows of SURVEY 8(f) through the C ABI against the oracle -- device-built maps (NEXT-2,
PAPER.md:108-133), the largest charge cluster and snapshots of the drop workload (NEXT-3)."""
import os

import numpy as np
import pytest

import ic_inputs
import oracle

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2301_11735_b200 as p
    return p


@pytest.mark.parametrize("L,bits,reps,K,nmaps", [(4, 8, 2, 3, 300), (16, 8, 3, 26, 200), (16, 2, 2, 60, 200), (64, 8, 3, 410, 120),
                                                 (64, 2, 2, 820, 60), (256, 8, 2, 6554, 40), (1024, 8, 1, 100000, 6),
                                                 (256, 2, 2, 6554, 40), (1024, 2, 1, 100000, 6)])   # 2 bits, L >= 128: layout P2
def test_map_sweeps_match_the_oracle(pkg, L, bits, reps, K, nmaps):
    """ic_sweep_maps: every map's candidates, survivors and pair updates equal the oracle's (mode 1), bit for bit: lattices,
    per-map integers, fp64 sums; sum S = Q after every map."""
    seed = 300 + L + bits
    nplus, nminus = L * L // 8, L * L // 16
    n = (nplus - nminus) / (L * L)
    Ts = [0.5, 1.2, 2.5][:reps]
    codes = [ic_inputs.random_state(L, nplus, nminus, seed, r) for r in range(reps)]
    sim = pkg.Sim(L, n, 0.3, 1.0, 1.5, seed=seed, replicas=reps, bits_per_site=bits)
    for r in range(reps):
        sim.set_state(r, codes[r])
    sim.sweep(Ts, 3)                                                     # maps continue a run of ordinary sweeps
    tr = sim.sweep_maps(Ts, nmaps, K, trace=True).cpu().numpy()
    assert sim.sweep_count == 3 + nmaps
    obs = sim.observables()
    for r in range(reps):
        lat = oracle.Lattice(codes[r], 0.3, 1.0, 1.5, seed, replica=r)
        lat.sweep_s1(Ts[r], 3)
        t, att = lat.sweep_maps(Ts[r], nmaps, 1, K, trace=True)
        assert att > 0
        assert np.array_equal(tr[:, r, :], t), f"per-map integers differ, replica {r}"
        assert (tr[:, r, 5] == sim.Q).all()
        assert np.array_equal(sim.state(r), lat.code)
        ref = lat.observables(Ts[r])
        for k in ("n2", "bV", "bJ", "M", "Ms", "Q", "nmeas", "sumE", "sumE2", "sumM2", "sumAbsMs"):
            assert obs[r][k] == ref[k], (r, k, obs[r][k], ref[k])
        assert np.array_equal(sim.debug_recompute(r), lat.ints())
    sim.close()


def test_map_sweeps_argument_checks(pkg):
    sim = pkg.Sim(16, 0.25, 0.5, 1.0, 1.0, seed=1)
    for bad in (lambda: sim.sweep_maps(1.0, 5, 0), lambda: sim.sweep_maps(0.0, 5, 10), lambda: sim.sweep_maps(1.0, -1, 10)):
        with pytest.raises(pkg.IcError):
            bad()
    assert sim.sweep_count == 0
    assert pkg.lib.ic_maps_scratch_bytes(16, 0) == 0 and pkg.lib.ic_cluster_scratch_bytes(24) == 0
    sim.close()


@pytest.mark.parametrize("L,bits,dens", [(4, 8, 0.5), (16, 8, 0.55), (16, 2, 0.3), (64, 8, 0.6), (64, 2, 0.45), (256, 8, 0.59), (2048, 8, 0.55),
                                         (256, 2, 0.59), (2048, 2, 0.55)])                            # 2 bits, L >= 128: layout P2
def test_largest_cluster_matches_the_oracle(pkg, L, bits, dens):
    """ic_largest_cluster (union-find on the device) against the oracle's flood fill, near the site-percolation threshold
    (0.593) where clusters are large and ragged; all three charge selections; two replicas."""
    N = L * L
    nplus, nminus = int(dens * N * 0.6), int(dens * N * 0.4)
    sim = pkg.Sim(L, (nplus - nminus) / N, 0.5, 1.0, 1.0, seed=4, replicas=2, bits_per_site=bits)
    for r in range(2):
        code = ic_inputs.random_state(L, nplus, nminus, 40 + L, r)
        sim.set_state(r, code)
        for which in (0, 1, 2):
            assert sim.largest_cluster(r, which) == oracle.largest_cluster(code, which), (r, which)
    sim.sweep([0.7, 1.4], 3)
    for r in range(2):
        assert sim.largest_cluster(r, 0) == oracle.largest_cluster(sim.state(r), 0)
    sim.close()
    for kind, want in (("all_plus", (N, 1)), ("ferro", (0, 0)), ("stripes", (N, 1))):
        code = ic_inputs.structured_state(L, kind)
        Q = int(np.array([0, 0, 1, -1])[code].sum())
        s2 = pkg.Sim(L, Q / N, 0.5, 1.0, 1.0, seed=1, bits_per_site=bits); s2.set_state(0, code)
        assert s2.largest_cluster(0, 0) == want
        s2.close()


def test_drop_workload_and_snapshot(pkg, tmp_path):
    """Config C6 (Fig. 7: J >> V, 64 x 64): quenched to a low temperature the charges gather into drops --
    the largest cluster of S=+1 sites is several times larger than at high temperature; trajectory and cluster sizes equal
    the oracle's; the PPM snapshot has one pixel per site in the documented colours."""
    c = ic_inputs.CONFIGS["C6"]
    L, Ts = c["L"], c["T"]
    sim = pkg.Sim(L, c["n"], c["delta"], c["V"], c["J"], seed=c["seed"], replicas=len(Ts))
    codes = [sim.state(r).copy() for r in range(len(Ts))]
    sim.sweep(Ts, c["sweeps"])
    sizes = []
    for r, T in enumerate(Ts):
        lat = oracle.Lattice(codes[r], c["delta"], c["V"], c["J"], c["seed"], replica=r)
        lat.sweep_s1(T, c["sweeps"], threads=4)
        assert np.array_equal(sim.state(r), lat.code)
        got = sim.largest_cluster(r, 1)
        assert got == oracle.largest_cluster(lat.code, 1)
        sizes.append(got[0])
    assert sizes[0] > 2.5 * sizes[-1] and sizes[0] >= 40, sizes        # the drop: a large part of the 410 charges in one cluster
    path = os.path.join(tmp_path, "drop.ppm")
    sim.snapshot_ppm(0, path)
    raw = open(path, "rb").read()
    head = b"P6\n%d %d\n255\n" % (L, L)
    assert raw.startswith(head) and len(raw) == len(head) + 3 * L * L
    px = np.frombuffer(raw[len(head):], dtype=np.uint8).reshape(L, L, 3)
    pal = np.array([[255, 255, 255], [64, 64, 64], [220, 30, 30], [30, 60, 220]], dtype=np.uint8)
    assert np.array_equal(px, pal[sim.state(0)])
    with pytest.raises(pkg.IcError):
        sim.snapshot_ppm(0, os.path.join(tmp_path, "no_such_dir", "x.ppm"))
    sim.close()
