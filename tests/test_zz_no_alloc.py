"""-m gpu: the entry point that allocates nothing (tpc_cf_scan_u32_static: the compaction's exclusive scan with its
scratch in a file-scope device array of the library) against the existing path (the same scan with its scratch in a
handle's caller-owned workspace) and against numpy, bit for bit, on two calls in a row — the second with other data
and another size, so that scratch left by the first call would show.  Collected last on purpose (file name): the
suite runs with pytest -x.  Must pass alone in a fresh process and after all other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _u32(t):
    return t.cpu().numpy().view(np.uint32)


def test_static_scratch_scan_matches_workspace_scan_two_calls_in_a_row():
    import torch
    import paper_2402_01205_b200 as cf
    lib = cf.load()
    dev = torch.device("cuda:0")
    torch.cuda.set_device(dev)
    limit = int(lib.tpc_cf_scan_static_max_n())
    assert limit == 1 << 26
    assert lib.tpc_cf_scan_static_setup() == 0            # once per device, with that device current
    finder = cf.ClusterFinder(1, 4, 16, 64, max_digits=1 << 16, max_clusters=64, sorted_only=True)
    rng = np.random.default_rng(2402)
    # two calls in a row; sizes span one block, many blocks + a ragged tail, and more partials than one scan block
    for n, hi in ((5_000_037, 1000), (1_234_567, 7), (1, 5), (1024, 4_000_000), (0, 1)):
        host = rng.integers(0, hi, size=max(n, 1), dtype=np.uint32)[:n]
        inp = torch.from_numpy(host.view(np.int32)).to(dev)
        out_new = torch.full((max(n, 1),), -1, dtype=torch.int32, device=dev)
        out_old = torch.full((max(n, 1),), -1, dtype=torch.int32, device=dev)
        tot_new = torch.full((1,), -1, dtype=torch.int64, device=dev)
        tot_old = torch.full((1,), -1, dtype=torch.int64, device=dev)
        before = torch.cuda.memory_allocated(dev)
        cf.scan_u32_static(inp, out_new, n, tot_new)
        assert torch.cuda.memory_allocated(dev) == before
        finder.debug_scan_u32(inp, out_old, n, tot_old)
        torch.cuda.synchronize()
        if n == 0:
            assert int(tot_new.item()) == 0
            continue
        want = np.zeros(n, dtype=np.uint64)
        np.cumsum(host[:-1].astype(np.uint64), out=want[1:])
        assert np.array_equal(_u32(out_new)[:n], (want & 0xffffffff).astype(np.uint32)), "static scan differs from numpy (n = %d)" % n
        assert np.array_equal(_u32(out_new)[:n], _u32(out_old)[:n]), "static scan differs from the workspace scan (n = %d)" % n
        assert int(tot_new.item()) == int(tot_old.item()) == int(host.astype(np.uint64).sum())
    # in place (in == out), as the library itself uses it
    host = rng.integers(0, 50, size=300_001, dtype=np.uint32)
    buf = torch.from_numpy(host.view(np.int32)).to(dev)
    cf.scan_u32_static(buf, buf, host.shape[0])
    torch.cuda.synchronize()
    assert np.array_equal(_u32(buf), np.concatenate([[0], np.cumsum(host[:-1].astype(np.uint64))]).astype(np.uint32))
    # beyond the static scratch: a clear error, nothing enqueued
    with pytest.raises(cf.TpcCfError) as e:
        cf.scan_u32_static(buf, buf, limit + 1)
    assert e.value.code == -3
    finder.close()
