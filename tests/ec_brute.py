"""Independent checker for the TPC-EC v1 container (test code; another language and other data structures than
oracle/tpc_ec_oracle.c, written from the format text in oracle/tpc_ec_oracle.h, not from the C code).

- lane_decode: the rANS decoding recurrence with the symbol found by numpy.searchsorted on the cumulative table
- parse / decode_container: struct-based container walk, clusters rebuilt with numpy cumulative sums per plane
- symbol_bytes: the (Q) streams of a cluster list computed with Python ints and numpy.float32 scalars
"""
import math
import struct

import numpy as np

L = 1 << 23
M = 4096
N_STREAMS, BLOCK, LANES = 13, 16384, 32


def lane_decode(state, data, freq, m):
    cum = np.concatenate([[0], np.cumsum(np.asarray(freq, dtype=np.int64))])
    x, ptr, out = int(state), len(data), []
    for _ in range(m):
        slot = x % M
        s = int(np.searchsorted(cum, slot, side="right")) - 1
        assert 0 <= s < 256 and freq[s] > 0
        out.append(s)
        x = int(freq[s]) * (x // M) + slot - int(cum[s])
        while x < L:
            assert ptr > 0, "lane ran out of bytes"
            ptr -= 1
            x = x * 256 + int(data[ptr])
    assert x == L and ptr == 0, (x, ptr)
    return out


def information_bits(symbols, freq):
    return sum(math.log2(M / int(freq[s])) for s in symbols)


def parse(buf):
    b = bytes(buf)
    magic, ver, n, n_sec, n_rows, n_str, blk, n_blocks, z, total = struct.unpack_from("<IIQIIIIIIQ", b, 0)
    assert magic == 0x45435054 and b[0:4] == b"TPCE" and ver == 1 and n_str == N_STREAMS and blk == BLOCK and z == 0
    assert n_blocks == (n + BLOCK - 1) // BLOCK and total == len(b) and b[48:64] == bytes(16)
    planes = n_sec * n_rows
    counts = np.frombuffer(b, dtype="<u4", count=planes, offset=64)
    off_freq = 64 + 4 * planes
    freq = np.frombuffer(b, dtype="<u2", count=N_STREAMS * 256, offset=off_freq).reshape(N_STREAMS, 256)
    end_freq = off_freq + 2 * 256 * N_STREAMS
    off_dir = (end_freq + 7) // 8 * 8
    assert b[end_freq:off_dir] == bytes(off_dir - end_freq)
    rec_off = np.frombuffer(b, dtype="<u8", count=N_STREAMS * n_blocks + 1, offset=off_dir)
    assert int(rec_off[-1]) == total
    if n_blocks:
        assert int(rec_off[0]) == off_dir + 8 * (N_STREAMS * n_blocks + 1)
    return dict(n=n, n_sectors=n_sec, n_rows=n_rows, n_blocks=n_blocks, counts=counts, freq=freq, rec_off=rec_off, raw=b)


def decode_streams(c):
    n, nb = c["n"], c["n_blocks"]
    streams = np.zeros((N_STREAMS, n), dtype=np.uint8)
    for s in range(N_STREAMS):
        for blk in range(nb):
            r0, r1 = int(c["rec_off"][s * nb + blk]), int(c["rec_off"][s * nb + blk + 1])
            rec = c["raw"][r0:r1]
            states = struct.unpack_from("<32I", rec, 0)
            nbytes = struct.unpack_from("<32H", rec, 128)
            at = 192
            for l in range(LANES):
                pos = np.arange(blk * BLOCK + l, min(n, (blk + 1) * BLOCK), LANES)
                streams[s, pos] = lane_decode(states[l], rec[at:at + nbytes[l]], c["freq"][s], len(pos))
                at += nbytes[l]
            pad = rec[at:]
            assert len(pad) < 4 and pad == bytes(len(pad)) and (r1 - r0) % 4 == 0
    return streams


def rebuild(c, streams, dtype):
    """inverse of (Q) with numpy: per plane, pads by cumulative sum, times by cumulative sum inside each pad line"""
    n = c["n"]
    out = np.zeros(n, dtype=dtype)
    st = streams.astype(np.int64)
    i = 0
    for pl, cnt in enumerate(c["counts"]):
        cnt = int(cnt)
        if cnt == 0:
            continue
        sl = slice(i, i + cnt)
        pad = np.cumsum(st[0, sl])
        v = st[1, sl] + 256 * st[2, sl]
        head = np.ones(cnt, dtype=bool)
        head[1:] = st[0, sl][1:] != 0
        seg = np.cumsum(head) - 1
        csum = np.cumsum(v)
        base = (csum - v)[head][seg]           # sum before the head of each element's pad line
        time = csum - base
        out["sector"][sl] = pl // c["n_rows"]
        out["row"][sl] = pl % c["n_rows"]
        out["pad"][sl] = pad
        out["time"][sl] = time
        i += cnt
    assert i == n
    qmax = st[3] + 256 * st[4]
    out["qmax"] = qmax
    out["qtot"] = qmax + st[5] + 256 * st[6] + 65536 * st[7]
    out["flags"] = st[8]
    out["pad_mean"] = out["pad"].astype(np.float64) + (st[9] - 128) / 64.0
    out["time_mean"] = out["time"].astype(np.float64) + (st[10] - 128) / 64.0
    out["sigma_pad"] = st[11] / 128.0
    out["sigma_time"] = st[12] / 128.0
    return out


def decode_container(buf, dtype):
    c = parse(buf)
    return rebuild(c, decode_streams(c), dtype)


def _q(v):
    v = np.float32(v)
    if np.isnan(v):
        return 0
    r = np.float32(np.rint(v))                 # round half to even
    return int(min(max(r, np.float32(0)), np.float32(255)))


def symbol_bytes(clusters, n_rows):
    """(Q) for a numpy cluster array, cluster by cluster."""
    n = len(clusters)
    out = np.zeros((N_STREAMS, n), dtype=np.uint8)
    f32 = np.float32
    for i, c in enumerate(clusters):
        p = clusters[i - 1] if i > 0 else None
        same = p is not None and (int(p["sector"]), int(p["row"])) == (int(c["sector"]), int(c["row"]))
        dpad = int(c["pad"]) - int(p["pad"]) if same else int(c["pad"])
        v = int(c["time"]) - int(p["time"]) if (same and dpad == 0) else int(c["time"])
        dq = (int(c["qtot"]) - int(c["qmax"])) % (1 << 24)
        out[0, i], out[1, i], out[2, i] = dpad, v % 256, v // 256
        out[3, i], out[4, i] = int(c["qmax"]) % 256, int(c["qmax"]) // 256
        out[5, i], out[6, i], out[7, i] = dq % 256, (dq // 256) % 256, dq // 65536
        out[8, i] = int(c["flags"])
        out[9, i] = _q(f32(f32(f32(c["pad_mean"]) - f32(int(c["pad"]))) + f32(2)) * f32(64))
        out[10, i] = _q(f32(f32(f32(c["time_mean"]) - f32(int(c["time"]))) + f32(2)) * f32(64))
        out[11, i] = _q(f32(c["sigma_pad"]) * f32(128))
        out[12, i] = _q(f32(c["sigma_time"]) * f32(128))
    return out
