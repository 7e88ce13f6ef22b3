"""-m "not gpu" tests of the boundary and the host logic: the C-ABI library loads and exports every symbol that
include/tpc_cf.h declares, workspace sizing, synchronous argument errors that need no device, the seeded generator's
contract (sorted, deterministic for any thread count, occupancies of BASELINE.json:configs), and the replica
sharding used for N > 1 under a world-size-2 gloo group.  No compute call is made here.
"""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header="tpc_cf.h", prefix="tpc_cf_"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(%s[a-z0-9_]+)\s*\(" % prefix, text)))


def test_library_exports_every_declared_symbol():
    import paper_2402_01205_b200 as cf
    lib = cf.load()
    syms = declared_symbols()
    assert "tpc_cf_create" in syms and "tpc_cf_run" in syms and "tpc_cf_destroy" in syms
    for s in syms:
        assert hasattr(lib, s), "libtpc_cf.so does not export %s" % s
    assert sorted(cf.EXPORTS) == syms, "binding.EXPORTS and include/tpc_cf.h disagree"


def test_every_header_under_include_is_covered():
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["tpc_cf.h", "tpc_ec.h", "tpc_fe.h"]


def test_library_exports_every_entropy_coder_symbol():
    import paper_2402_01205_b200 as cf
    lib = cf.load()
    syms = declared_symbols("tpc_ec.h", "tpc_ec_")
    assert "tpc_ec_encode" in syms and "tpc_ec_decode" in syms
    for s in syms:
        assert hasattr(lib, s), "libtpc_cf.so does not export %s" % s
    assert sorted(cf.EC_EXPORTS) == syms, "ec_binding.EC_EXPORTS and include/tpc_ec.h disagree"
    src = open(os.path.join(ROOT, "paper_2402_01205_b200", "ec_binding.py")).read()
    assert "oracle" not in src, "the product binding must not reference the oracle"


def test_library_exports_every_front_end_filter_symbol():
    import paper_2402_01205_b200 as cf
    lib = cf.load()
    syms = declared_symbols("tpc_fe.h", "tpc_fe_")
    assert "tpc_fe_create" in syms and "tpc_fe_run" in syms and "tpc_fe_destroy" in syms
    for s in syms:
        assert hasattr(lib, s), "libtpc_cf.so does not export %s" % s
    assert sorted(cf.FE_EXPORTS) == syms, "fe_binding.FE_EXPORTS and include/tpc_fe.h disagree"
    src = open(os.path.join(ROOT, "paper_2402_01205_b200", "fe_binding.py")).read()
    assert "oracle" not in src, "the product binding must not reference the oracle"
    src = open(os.path.join(ROOT, "paper_2402_01205_b200", "csrc", "tpc_fe.cu")).read()
    assert "#include \"../../oracle" not in src and "tpc_fe_oracle.h" not in src


def test_front_end_filter_host_logic_without_a_device():
    """sizes and the synchronous argument errors of include/tpc_fe.h that are decided before any device call"""
    import paper_2402_01205_b200 as cf
    from paper_2402_01205_b200 import fe_binding as fb
    assert cf.FE_STATUS.itemsize == 16 and ctypes.sizeof(cf.FeParams) == 8
    assert [cf.tpc_fe_pad_stride(p) for p in (1, 8, 9, 138, 255)] == [8, 8, 16, 144, 256]
    g, keep = cf.make_geometry(36, 152, 138, 14336)
    w = cf.tpc_fe_workspace_bytes(g, 65536)
    planes = 36 * 152
    fixed = 4 * planes * 65536 + 4 * planes * 2048 + 4 * planes * 144      # records, chunk directory, line counts
    assert fixed < w < fixed + 80 * planes + 4096
    assert cf.tpc_fe_workspace_bytes(g, 0) == 0 and cf.tpc_fe_workspace_bytes(g, 1 << 32) == 0
    bad, _ = cf.make_geometry(36, 152, 256, 14336)
    assert cf.tpc_fe_workspace_bytes(bad, 100) == 0
    lib = fb._lib()
    h = ctypes.c_void_p()
    fake = ctypes.c_void_p(1 << 20)
    assert lib.tpc_fe_create(ctypes.byref(h), ctypes.byref(g), 65536, None, w) == -1
    assert lib.tpc_fe_create(ctypes.byref(h), ctypes.byref(bad), 65536, fake, w) == -2
    assert lib.tpc_fe_create(ctypes.byref(h), ctypes.byref(g), 0, fake, w) == -3
    assert lib.tpc_fe_create(ctypes.byref(h), ctypes.byref(g), 65536, ctypes.c_void_p((1 << 20) + 8), w) == -4
    assert lib.tpc_fe_create(ctypes.byref(h), ctypes.byref(g), 65536, fake, 1000) == -4
    assert lib.tpc_fe_destroy(None) == -1
    with pytest.raises(RuntimeError):
        import torch
        if torch.cuda.is_available():
            raise RuntimeError("device present: the no-fallback check is for CPU boxes")
        cf.FrontEndFilter(1, 1, 8, 64)


def test_entropy_coder_host_logic_without_a_device():
    """sizes and synchronous argument errors of include/tpc_ec.h (no kernel is launched: create / destroy keep host
    state only, and every check below fails before the first enqueue)"""
    import paper_2402_01205_b200 as cf
    from paper_2402_01205_b200 import ec_binding as eb
    assert cf.EC_STATUS.itemsize == 24
    assert cf.tpc_ec_workspace_bytes(0, 152, 100) == 0 and cf.tpc_ec_workspace_bytes(36, 257, 100) == 0
    assert cf.tpc_ec_workspace_bytes(36, 152, 1 << 32) == 0
    w = cf.tpc_ec_workspace_bytes(36, 152, 12_000_000)
    # 13 symbol bytes per cluster + the lanes' worst-case slots (13 * 32 * 776 bytes per block of 16384 clusters)
    assert 32 * 12_000_000 < w < 34 * 12_000_000 + (1 << 20)
    # fixed part of the container: header, plane counts, 13 tables, directory; then <= 12 bits per symbol + slack
    n = 100_000
    nb = (n + 16383) // 16384
    fixed = ((64 + 4 * 36 * 152 + 2 * 256 * 13 + 7) & ~7) + 8 * (13 * nb + 1)
    m = cf.tpc_ec_max_encoded_bytes(36, 152, n)
    assert fixed + 13 * n * 3 // 2 <= m <= fixed + 13 * n * 3 // 2 + 13 * nb * 300
    assert cf.tpc_ec_max_encoded_bytes(36, 152, 0) == fixed - 8 * 13 * nb
    lib = eb._lib()
    h = ctypes.c_void_p()
    fake = ctypes.c_void_p(1 << 20)                                   # never dereferenced by the calls below
    assert lib.tpc_ec_create(ctypes.byref(h), 36, 152, 1000, None, w) == -1
    assert lib.tpc_ec_create(ctypes.byref(h), 0, 152, 1000, fake, w) == -2
    assert lib.tpc_ec_create(ctypes.byref(h), 36, 152, 1000, ctypes.c_void_p((1 << 20) + 8), w) != 0   # misaligned
    assert lib.tpc_ec_create(ctypes.byref(h), 36, 152, 1000, fake, 1000) != 0                         # too small
    assert lib.tpc_ec_create(ctypes.byref(h), 36, 152, 1000, fake, w) == 0
    assert lib.tpc_ec_encode(h, fake, 1001, fake, 1 << 30, fake, None) != 0       # n > max_clusters
    assert lib.tpc_ec_encode(h, fake, 10, None, 1 << 30, fake, None) == -1        # NULL out
    assert lib.tpc_ec_encode(h, fake, 10, fake, 100, fake, None) != 0             # below the fixed part
    assert lib.tpc_ec_encode(h, fake, 10, ctypes.c_void_p((1 << 20) + 4), 1 << 30, fake, None) != 0   # misaligned
    assert lib.tpc_ec_decode(h, fake, 40, 10, fake, 10, fake, None) != 0          # shorter than the fixed part
    assert lib.tpc_ec_decode(h, None, 1 << 20, 10, fake, 10, fake, None) == -1
    assert lib.tpc_ec_destroy(h) == 0
    assert lib.tpc_ec_destroy(None) == -1


def test_library_is_sm100a_and_uses_no_fallback():
    import paper_2402_01205_b200 as cf
    from paper_2402_01205_b200 import build
    cf.load()
    out = subprocess.run(["cuobjdump", "-lelf", build.SO], capture_output=True, text=True)
    if out.returncode == 0:
        assert "sm_100a" in out.stdout, out.stdout
    # no file of the product package may name the oracle in code, in any spelling (import, include, path, dlopen of
    # its library); comments of the C/CUDA sources may say that nothing is shared with it
    import re
    pkg = os.path.join(ROOT, "paper_2402_01205_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            path = os.path.join(dirpath, fn)
            if fn.endswith(".py"):
                src = open(path, errors="replace").read().lower()
            elif fn.endswith((".cu", ".cuh", ".h", ".c", ".cpp")):
                src = open(path, errors="replace").read().lower()
                src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)
                src = re.sub(r"//[^\n]*", " ", src)
            else:
                continue
            assert "oracle" not in src, "the product must not reference the oracle: %s" % path
    binding = open(os.path.join(pkg, "binding.py")).read()
    assert "oracle" not in binding.lower()


def test_struct_layouts_match_header():
    import paper_2402_01205_b200 as cf
    assert cf.DIGIT.itemsize == 8 and cf.CLUSTER.itemsize == 32 and cf.STATUS.itemsize == 32
    assert cf.CLUSTER.fields["qtot"][1] == 8 and cf.CLUSTER.fields["pad_mean"][1] == 12
    assert ctypes.sizeof(cf.Geometry) == 24 and ctypes.sizeof(cf.Params) == 16 and ctypes.sizeof(cf.Out) == 32


def test_variant_bits_agree_between_header_binding_and_oracle_header():
    """bench.py and the GPU tests pass the same flag word to the library and to the oracle: the enumerators of
    include/tpc_cf.h, the constants of the binding and the (independently written) oracle header must agree."""
    import re
    root = os.path.join(os.path.dirname(__file__), "..")
    hdr = open(os.path.join(root, "include", "tpc_cf.h")).read()
    orc_hdr = open(os.path.join(root, "oracle", "tpc_cf_oracle.h")).read()

    def enum(text, name):
        m = re.search(r"\b%s\s*=\s*(\d+)u?" % name, text)
        assert m, name
        return int(m.group(1))
    from paper_2402_01205_b200 import binding
    from oracle import oracle as orc
    for name in ("CLUSTER_FLAGS", "CUT_SINGLE_PAD", "CUT_SINGLE_TIME", "SHARE_CHARGE"):
        assert enum(hdr, "TPC_CF_" + name) == getattr(binding, name) == getattr(orc, name) == enum(orc_hdr, "ORC_" + name)
    for name in ("EDGE_PAD", "EDGE_TIME", "SINGLE_PAD", "SINGLE_TIME", "SATURATED", "SHARED"):
        assert (enum(hdr, "TPC_CF_F_" + name) == getattr(binding, "F_" + name) == getattr(orc, "F_" + name)
                == enum(orc_hdr, "ORC_F_" + name))


def test_workspace_bytes_and_geometry_limits():
    import paper_2402_01205_b200 as cf
    g, _ = cf.make_geometry(36, 152, 138, 14336)
    full = cf.tpc_cf_workspace_bytes(g, 220_000_000, 14_000_000)
    # dense uint16 map with a 2-cell border dominates: 36*152 planes x 142 x 14344 cells
    map_bytes = 36 * 152 * 142 * 14344 * 2
    assert full > map_bytes and full < map_bytes + 220_000_000 * 40 + 14_000_000 * 64 + (1 << 26)
    small = cf.tpc_cf_workspace_bytes(g, 1000, 100)
    assert map_bytes < small < full
    for bad in ((0, 152, 138, 14336), (36, 0, 138, 14336), (36, 152, 256, 14336), (36, 152, 138, 65536),
                (257, 152, 138, 14336)):
        gb, _ = cf.make_geometry(*bad)
        assert cf.tpc_cf_workspace_bytes(gb, 1000, 100) == 0
    gn, keep = cf.make_geometry(1, 3, 16, 64, npads=[10, 17, 16])       # 17 > max_pads
    assert cf.tpc_cf_workspace_bytes(gn, 10, 10) == 0
    assert cf.tpc_cf_workspace_bytes(g, 1 << 32, 10) == 0                # capacities must stay below 2^32


def test_synchronous_errors_without_a_device():
    import paper_2402_01205_b200 as cf
    lib = cf.load()
    g, _ = cf.make_geometry(1, 2, 8, 16)
    h = ctypes.c_void_p()
    assert lib.tpc_cf_create(ctypes.byref(h), ctypes.byref(g), 10, 10, None, 0, None) == -1          # E_NULL
    buf = ctypes.create_string_buffer(1 << 16)
    addr = (ctypes.addressof(buf) + 255) & ~255
    assert lib.tpc_cf_create(ctypes.byref(h), ctypes.byref(g), 10, 10, addr + 8, 1 << 15, None) == -4  # misaligned
    assert lib.tpc_cf_create(ctypes.byref(h), ctypes.byref(g), 10, 10, addr, 64, None) == -4           # too small
    gb, _ = cf.make_geometry(0, 2, 8, 16)
    assert lib.tpc_cf_create(ctypes.byref(h), ctypes.byref(gb), 10, 10, addr, 1 << 15, None) == -2     # E_GEOMETRY
    assert lib.tpc_cf_run(None, None, 0, ctypes.byref(g), None, None) == -1
    assert lib.tpc_cf_destroy(None) == -1
    for code in range(-7, 1):
        assert lib.tpc_cf_strerror(code)
    assert b"unknown" in lib.tpc_cf_strerror(-99)


def test_product_fails_loudly_without_cuda():
    import torch
    import paper_2402_01205_b200 as cf
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        cf.ClusterFinder(1, 2, 8, 16, max_digits=16)


# ---- generator ---------------------------------------------------------------------------------------------------

def digit_keys(d):
    return ((d["sector"].astype(np.uint64) << 32) | (d["row"].astype(np.uint64) << 24) |
            (d["pad"].astype(np.uint64) << 16) | d["time"].astype(np.uint64))


def test_generator_contract_config1():
    from datagen import gen
    d1 = gen.generate(1, n_threads=1)
    d4 = gen.generate(1, n_threads=4)
    assert np.array_equal(d1, d4), "output depends on the thread count"
    k = digit_keys(d1)
    assert np.all(k[1:] > k[:-1]), "digits not strictly ascending in (sector,row,pad,time) / duplicate cells"
    assert d1["charge"].min() >= 2 and d1["time"].max() < 512 and d1["pad"].max() < 138 and d1["row"].max() < 152
    assert 0.004 < gen.occupancy(d1, 1) < 0.008                       # config 1 comes out ~0.57 %
    assert gen.checksum(d1) == gen.checksum(d4)
    part = gen.generate(dict(gen.CONFIGS[3], n_sectors=36), sectors=(5, 6))
    assert part["sector"].min() == 5 and part["sector"].max() == 5


@pytest.mark.parametrize("cfg,lo,hi", [(2, 0.045, 0.055), (3, 0.018, 0.022), (4, 0.09, 0.11), (5, 0.0045, 0.0055)])
def test_generator_occupancies(cfg, lo, hi):
    """±10 % of the occupancies BASELINE.json:configs states, measured on one sector."""
    from datagen import gen
    c = dict(gen.CONFIGS[cfg], n_sectors=1)
    d = gen.generate(c)
    assert lo < gen.occupancy(d, c) < hi
    k = digit_keys(d)
    assert np.all(k[1:] > k[:-1])
    if cfg == 5:
        npads = gen.geometry(c)[4]
        assert npads[0] == 66 and npads[-1] == 138 and int(npads.sum()) == 15429
        assert np.all(d["pad"] < npads[d["row"]])


def test_generator_plateaus_yield_one_peak_each():
    """config 4 injects rectangular flat tops (R1b): the oracle must find exactly one peak per plateau cell set,
    at its (min pad, min time) corner — checked on the plateau cells that are still flat in the output."""
    from datagen import gen
    from oracle import oracle as orc
    c = dict(gen.CONFIGS[4], n_sectors=1, n_rows=4)
    d = gen.generate(c)
    cl, st = orc.run(d, 1, 4, 138, 14336)
    assert st["n_clusters"] > 1000
    # a peak's later neighbour in time never exceeds it, and equal-charge horizontal runs start at the peak
    peaks = {(int(x["row"]), int(x["pad"]), int(x["time"])): int(x["qmax"]) for x in cl}
    cells = {(int(x["row"]), int(x["pad"]), int(x["time"])): int(x["charge"]) for x in d[d["row"] == 0]}
    flat_pairs = 0
    for (r, p, t), q in cells.items():
        if q >= 30 and cells.get((r, p, t + 1)) == q:
            flat_pairs += 1
            assert (r, p, t + 1) not in peaks, "second cell of a flat run must not be a peak"
    assert flat_pairs > 0


# ---- N > 1: replicas only ------------------------------------------------------------------------

_GLOO_WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import numpy as np
import torch, torch.distributed as dist
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
from datagen import gen
from oracle import oracle as orc
cfg = dict(gen.CONFIGS[1])
# replicas: rank r owns frame r; value = sum of units / max of times, exactly as bench.py aggregates
d = gen.generate(cfg, frame=rank)
cl, st = orc.run(d, *gen.geometry(cfg)[:4])
t = torch.tensor([10.0 + rank], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
c = torch.tensor([float(d.shape[0]), float(st["n_clusters"])], dtype=torch.float64)
dist.all_reduce(c, op=dist.ReduceOp.SUM)
if rank == 0:
    print(json.dumps({"tmax": t.item(), "digits": c[0].item(), "clusters": c[1].item(), "own": int(d.shape[0])}))
dist.barrier()
dist.destroy_process_group()
"""


def test_replica_sharding_world_size_2_gloo(tmp_path):
    """Frames go round-robin to ranks with no data-path collective; the only collectives are the
    timing MAX and the unit SUM that bench.py uses.  Run with the gloo backend on CPU, world size 2."""
    from datagen import gen
    port = 29500 + (os.getpid() % 2000)
    script = tmp_path / "worker.py"
    script.write_text(_GLOO_WORKER % {"root": ROOT, "port": port})
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    import json
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    n0 = gen.generate(1, frame=0).shape[0]
    n1 = gen.generate(1, frame=1).shape[0]
    assert res["tmax"] == 11.0 and res["digits"] == n0 + n1 and res["own"] == n0 and n0 != n1


# ---- N > 1, latency mode: one frame cut into plane ranges -------------------------------

def test_plane_partition_is_contiguous_complete_and_balanced():
    import paper_2402_01205_b200 as cf
    from datagen import gen
    c = dict(gen.CONFIGS[1])
    d = gen.generate(c)
    ns, nr = c["n_sectors"], c["n_rows"]
    ps = cf.plane_counts(d, ns, nr)
    assert ps.shape == (ns * nr + 1,) and ps[0] == 0 and ps[-1] == d.shape[0] and np.all(np.diff(ps) >= 0)
    key = d["sector"].astype(np.int64) * nr + d["row"]
    assert np.array_equal(np.diff(ps), np.bincount(key, minlength=ns * nr))
    biggest = int(np.diff(ps).max())
    for world in (1, 2, 3, 8, 200):
        part = cf.plane_partition(ps, world)
        assert len(part) == world and part[0][0] == 0 and part[-1][1] == ns * nr
        for a, b in zip(part, part[1:]):
            assert a[1] == b[0] and a[3] == b[2]                          # contiguous in planes and in digits
        for (pb, pe, db, de) in part:
            assert pb <= pe and db == ps[pb] and de == ps[pe]
            assert de - db <= d.shape[0] // world + biggest + 1            # balanced up to one plane
    # degenerate inputs: no digits at all, everything in one plane
    assert cf.plane_partition(np.zeros(11, dtype=np.int64), 3)[-1][1] == 10
    one = np.zeros(11, dtype=np.int64)
    one[4:] = 1000
    part = cf.plane_partition(one, 4)
    assert sum(p[3] - p[2] for p in part) == 1000 and max(p[3] - p[2] for p in part) == 1000


_SHARD_WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import numpy as np
import torch, torch.distributed as dist
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%(port)d", rank=int(sys.argv[1]), world_size=2)
rank = dist.get_rank()
from datagen import gen
from oracle import oracle as orc
from paper_2402_01205_b200.shard import plane_counts, plane_partition, gather_records
cfg = dict(gen.CONFIGS[1])
g = gen.geometry(cfg)
d = gen.generate(cfg)
part = plane_partition(plane_counts(d, g[0], g[1]), 2)[rank]
# the rank's compute step: here the CPU oracle stands in for the CUDA cluster finder (no GPU in this test)
mine = d[part[2]:part[3]]
cl, st = orc.run(mine, *g[:4], planes=(part[0], part[1]))
local = torch.from_numpy(cl.view(np.uint8).copy())
out, counts = gather_records(local, cl.shape[0], 32, 0)
if rank == 0:
    whole, wst = orc.run(d, *g[:4])
    same = out.numpy().tobytes() == whole.tobytes()
    print(json.dumps({"same": bool(same), "counts": counts, "total": int(wst["n_clusters"]), "part": list(part)}))
else:
    assert out is None
dist.barrier()
dist.destroy_process_group()
"""


def test_sector_sharded_frame_world_size_2_gloo(tmp_path):
    """Latency mode: the frame's planes are cut into two contiguous ranges balanced by digit count, every rank
    processes its slice alone, and the variable-size gather in rank order gives exactly the single-rank result
    (planes are independent, R2).  gloo backend on CPU; the oracle stands in for the per-rank CUDA step."""
    port = 31500 + (os.getpid() % 2000)
    script = tmp_path / "shard_worker.py"
    script.write_text(_SHARD_WORKER % {"root": ROOT, "port": port})
    procs = [subprocess.Popen([sys.executable, str(script), str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                              text=True) for r in range(2)]
    outs = [p.communicate(timeout=300) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e[-2000:]
    import json
    res = json.loads(outs[0][0].strip().splitlines()[-1])
    assert res["same"] and sum(res["counts"]) == res["total"] and min(res["counts"]) > 0.4 * res["total"]


# ---- bench.py's reference arm (the oracle timed on the host cores) runs without a GPU ------------------------------

@pytest.mark.parametrize("stage,metric,unit", [("cf", "tpc_digits_per_second", "digits/s"),
                                               ("fe", "tpc_raw_samples_filtered_per_second", "samples/s"),
                                               ("ec", "tpc_clusters_encoded_per_second", "clusters/s")])
def test_bench_reference_arm_prints_one_json_line(stage, metric, unit):
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--stage", stage,
                          "--config", "1", "--steps", "1", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["metric"] == metric and j["unit"] == unit and j["value"] > 0
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] == 1
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["e2e"]["d2h_bytes_per_step"] == 0


def test_bench_product_arm_refuses_to_run_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    for extra in ([], ["--stage", "fe"], ["--stage", "ec"], ["--stage", "chain"]):
        out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--config", "1", "--steps", "1"] + extra,
                             capture_output=True, text=True, timeout=300)
        assert out.returncode != 0 and "no CPU fallback" in out.stderr
