"""GPU parity tests of the front-end filter (include/tpc_fe.h, csrc/tpc_fe.cu) against the oracle
(oracle/tpc_fe_oracle.c): bit-exact digit arrays (integer work) on the same seeded raw samples, through the C ABI."""
import numpy as np
import pytest

from datagen import gen, fe_gen
from oracle import fe_oracle as feo

pytestmark = pytest.mark.gpu


def _cf():
    import paper_2402_01205_b200 as cf
    return cf


def gpu_run(raw, ped4, ns, nr, mp, nt, npads=None, cap_plane=None, capacity=None, flt=None, **prm):
    import torch
    cf = _cf()
    own = flt is None
    if own:
        flt = cf.FrontEndFilter(ns, nr, mp, nt, npads=npads,
                                max_digits_per_plane=cap_plane if cap_plane else (nt + 32) * ((mp + 31) // 32 * 32))   # can never overflow
    r = torch.from_numpy(np.ascontiguousarray(raw).view(np.int16)).cuda()
    p = torch.from_numpy(np.ascontiguousarray(ped4).view(np.int16)).cuda()
    cap = capacity if capacity is not None else ns * nr * nt * mp
    out = torch.zeros(max(cap, 1) * 8, dtype=torch.uint8, device="cuda:0")
    flt.run(r, p, out, capacity=cap, **prm)
    st = flt.read_status()
    n = min(st["n_digits"], cap)
    d = out[:n * 8].cpu().numpy().view(cf.DIGIT)
    if own:
        flt.close()
    return d, st


def check(raw, ped4, ns, nr, mp, nt, npads=None, **prm):
    want, wst = feo.run(raw, ped4, ns, nr, mp, nt, npads=npads, capacity=ns * nr * nt * mp, **prm)
    got, st = gpu_run(raw, ped4, ns, nr, mp, nt, npads=npads, **prm)
    assert st == {"n_digits": wst["n_digits"], "overflow": 0}
    assert got.tobytes() == want.tobytes()
    return want


def random_raw(rng, ns, nr, mp, nt, p_spike=0.05):
    W = feo.pad_stride(mp)
    ped4 = rng.integers(100, 400, size=(ns * nr, W)).astype(np.uint16)
    base = rng.integers(20, 110, size=(ns * nr, nt, W))
    spikes = (rng.random((ns * nr, nt, W)) < p_spike) * rng.integers(0, 3000, size=(ns * nr, nt, W))
    return (base + spikes).astype(np.uint16), ped4


def test_hand_example_on_the_gpu():
    raw = np.full((1, 4, 8), 0xFFFF, dtype=np.uint16)
    raw[0, :, :3] = [[10, 10, 30], [8, 9, 12], [10, 10, 10], [10, 12, 9]]
    ped4 = np.full((1, 8), 0xFFFF, dtype=np.uint16)
    ped4[0, :3] = [40, 41, 38]
    got, st = gpu_run(raw, ped4, 1, 1, 3, 4, zs_threshold=2, cm_quiet4=8, cm_min_pads=2, it_decay_shift=1,
                      it_kappa_shift=2)
    assert [(int(d["pad"]), int(d["time"]), int(d["charge"])) for d in got] == [(2, 0, 21), (2, 1, 9), (2, 2, 5), (2, 3, 3)]


@pytest.mark.parametrize("mp,nt,ns,nr", [(1, 1, 1, 1), (7, 63, 1, 2), (8, 64, 2, 1), (33, 65, 1, 3), (138, 200, 1, 3),
                                         (100, 129, 2, 2), (255, 130, 1, 2), (160, 257, 1, 1), (200, 64, 1, 2),
                                         (60, 1000, 1, 5), (96, 70, 1, 2), (223, 77, 1, 1)])
def test_random_shapes_bit_exact(mp, nt, ns, nr):
    """every warp count (1..8 warps per plane), ragged last tiles, several tiles, single cells"""
    rng = np.random.default_rng(mp * 1000 + nt)
    raw, ped4 = random_raw(rng, ns, nr, mp, nt)
    k = int(rng.integers(1, 8))
    check(raw, ped4, ns, nr, mp, nt, zs_threshold=int(rng.integers(1, 5)), cm_quiet4=int(rng.integers(0, 80)),
          cm_min_pads=int(rng.integers(1, 6)), it_decay_shift=k, it_kappa_shift=int(rng.integers(k, 15)))


def test_parameter_corners_and_saturation():
    rng = np.random.default_rng(77)
    ns, nr, mp, nt = 1, 2, 40, 150
    raw, ped4 = random_raw(rng, ns, nr, mp, nt, p_spike=0.2)
    raw[0, 50:, 3] = 65535                     # saturating charge, the largest tail state
    raw[1, :, :] = 0                           # all samples below the pedestal
    for prm in (dict(zs_threshold=1, cm_quiet4=4095, cm_min_pads=1, it_decay_shift=14, it_kappa_shift=14),
                dict(zs_threshold=65535, cm_quiet4=0, cm_min_pads=1, it_decay_shift=1, it_kappa_shift=1),
                dict(zs_threshold=2, cm_quiet4=12, cm_min_pads=60000, it_decay_shift=6, it_kappa_shift=0),
                dict(zs_threshold=1, cm_quiet4=300, cm_min_pads=40, it_decay_shift=1, it_kappa_shift=14)):
        check(raw, ped4, ns, nr, mp, nt, **prm)


def test_variable_pads_per_row_and_poisoned_padding():
    rng = np.random.default_rng(5)
    ns, nr, mp, nt = 2, 6, 138, 140
    npads = np.array([66, 80, 1, 138, 97, 129], dtype=np.uint16)
    raw, ped4 = random_raw(rng, ns, nr, mp, nt)
    for r in range(nr):
        raw[r::nr, :, int(npads[r]):] = 0xFFFF
        ped4[r::nr, int(npads[r]):] = 0xFFFF
    want = check(raw, ped4, ns, nr, mp, nt, npads=npads, zs_threshold=2, cm_quiet4=40, cm_min_pads=3,
                 it_decay_shift=4, it_kappa_shift=6)
    assert np.all(want["pad"] < npads[want["row"]])


def test_generated_frame_config1_defaults_and_chain_into_the_cluster_finder():
    """BASELINE.json configs[0] as raw samples (forward model of datagen/fe_gen.py): filter on the device, digits equal
    to the oracle's, then straight into the cluster finder on the device (the chain of PAPER.md:57)"""
    import torch
    cf = _cf()
    g = gen.geometry(1)
    d = gen.generate(1)
    raw, ped4 = fe_gen.raw_from_digits(d, *g[:4], npads=g[4], seed=11)
    want, wst = feo.run(raw, ped4, *g[:4], npads=g[4], zs_threshold=3)
    flt = cf.FrontEndFilter(*g[:4], npads=g[4], max_digits_per_plane=8192)
    r = torch.from_numpy(raw.view(np.int16)).cuda()
    p = torch.from_numpy(ped4.view(np.int16)).cuda()
    out = torch.zeros(want.shape[0] * 8 + 800, dtype=torch.uint8, device="cuda:0")
    flt.run(r, p, out, zs_threshold=3)
    st = flt.read_status()
    assert st == {"n_digits": wst["n_digits"], "overflow": 0}
    n = st["n_digits"]
    assert out[:n * 8].cpu().numpy().tobytes() == want.tobytes()
    assert 0.5 * d.shape[0] < n < 1.2 * d.shape[0]
    # chain: the filter's digits are the cluster finder's input, in place on the device, and pass its order check
    finder = cf.ClusterFinder(*g[:4], npads=g[4], max_digits=n, max_clusters=n // 4)
    finder.run(out, n, flags=cf.DIGITS_SORTED)
    cl, cst = finder.result()
    assert cst["path"] == 3 and cst["n_bad_digits"] == 0 and cst["n_clusters"] > 1000
    from oracle import oracle as orc
    ocl, ost = orc.run(want, *g[:4], npads=g[4])
    assert ost["n_clusters"] == cst["n_clusters"]
    for f in ("sector", "row", "pad", "time", "qmax", "qtot"):
        assert np.array_equal(cl[f], ocl[f]), f
    finder.close()
    flt.close()


@pytest.mark.parametrize("cfg_id", [3, 4, 5])
def test_full_length_planes_in_the_bench_configuration(cfg_id):
    """the launch configuration bench.py --stage fe times (n_time 14336, 138 pads; config 3's ~2 %, config 4's ~10 % with
    close pairs and plateaus, config 5's pads 66 -> 138), a handle reused for two runs, against the oracle on every
    record"""
    import torch
    cf = _cf()
    c = dict(gen.CONFIGS[cfg_id])
    c["n_sectors"], c["n_rows"] = 1, 6
    ns, nr, mp, nt, npads = gen.geometry(c)
    d = gen.generate(c)
    raw, ped4 = fe_gen.raw_from_digits(d, ns, nr, mp, nt, npads=npads, seed=3)
    want, wst = feo.run(raw, ped4, ns, nr, mp, nt, npads=npads, zs_threshold=3)
    flt = cf.FrontEndFilter(ns, nr, mp, nt, npads=npads, max_digits_per_plane=1 << 19)
    for _ in range(2):
        got, st = gpu_run(raw, ped4, ns, nr, mp, nt, npads=npads, flt=flt, zs_threshold=3)
        assert st == {"n_digits": wst["n_digits"], "overflow": 0} and got.tobytes() == want.tobytes()
    flt.close()
    assert 0.6 * d.shape[0] < want.shape[0] < 1.1 * d.shape[0]


def test_overflow_bits_and_true_count():
    rng = np.random.default_rng(8)
    ns, nr, mp, nt = 1, 3, 50, 200
    raw, ped4 = random_raw(rng, ns, nr, mp, nt, p_spike=0.1)
    prm = dict(zs_threshold=2, cm_quiet4=12, cm_min_pads=8, it_decay_shift=6, it_kappa_shift=8)
    want, wst = feo.run(raw, ped4, ns, nr, mp, nt, **prm)
    n = wst["n_digits"]
    # output capacity too small: true count, bit 2, and the records below the capacity are the oracle's first ones
    got, st = gpu_run(raw, ped4, ns, nr, mp, nt, capacity=n // 2, **prm)
    assert st == {"n_digits": n, "overflow": 2} and got.tobytes() == want[:n // 2].tobytes()
    # staging too small: true count and bit 1
    got, st = gpu_run(raw, ped4, ns, nr, mp, nt, cap_plane=10, **prm)
    assert st["n_digits"] == n and st["overflow"] & 1


def test_synchronous_errors():
    import torch
    cf = _cf()
    flt = cf.FrontEndFilter(1, 1, 8, 64)
    r = torch.zeros(64 * 8, dtype=torch.int16, device="cuda:0")
    p = torch.zeros(8, dtype=torch.int16, device="cuda:0")
    out = torch.zeros(64 * 8 * 8, dtype=torch.uint8, device="cuda:0")
    for bad in (dict(zs_threshold=0), dict(cm_quiet4=4096), dict(cm_min_pads=0), dict(it_decay_shift=0),
                dict(it_decay_shift=9, it_kappa_shift=8)):
        with pytest.raises(cf.TpcCfError):
            flt.run(r, p, out, **bad)
    with pytest.raises(ValueError):
        flt.run(r[:100], p, out)
    flt.run(r, p, out)
    assert flt.read_status() == {"n_digits": 0, "overflow": 0} and flt.last_launch_count() == 3
    flt.close()
