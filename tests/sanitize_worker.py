"""Child process of tests/test_sanitizers.py: runs the three oracles and the two input generators from libraries built
with -fsanitize=address,undefined (the parent sets LD_PRELOAD to the sanitizer runtimes and passes the directory that
holds the instrumented libraries).  Prints one JSON line of counts / checksums; a sanitizer report aborts the process."""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
libdir = sys.argv[1] if len(sys.argv) > 1 and sys.argv[1] != "-" else None

from datagen import gen, fe_gen                      # noqa: E402
from oracle import oracle as orc, ec_oracle, fe_oracle   # noqa: E402

if libdir:
    gen._SO = os.path.join(libdir, "libtpc_gen.so")
    fe_gen._SO = os.path.join(libdir, "libtpc_fe_gen.so")
    orc._SO = os.path.join(libdir, "libtpc_cf_oracle.so")
    ec_oracle._SO = os.path.join(libdir, "libtpc_ec_oracle.so")
    fe_oracle._SO = os.path.join(libdir, "libtpc_fe_oracle.so")

out = {}
# cluster finder oracle: config 1, a dense slice with pairs and plateaus, variable pads, variants, edge inputs
d1 = gen.generate(1)
g1 = gen.geometry(1)
cl1, st1 = orc.run(d1, *g1[:4])
out["c1"] = [int(d1.shape[0]), "%016x" % gen.checksum(d1), st1["n_clusters"], int(cl1["qtot"].astype(np.uint64).sum())]
c4 = dict(gen.CONFIGS[4]); c4["n_sectors"] = 1; c4["n_rows"] = 3
d4 = gen.generate(c4)
cl4, st4 = orc.run(d4, *gen.geometry(c4)[:4], flags=4 | 8, q_tot_min=30, q_saturation=100)
out["c4"] = [int(d4.shape[0]), st4["n_clusters"], int(cl4["flags"].astype(np.uint64).sum())]
c5 = dict(gen.CONFIGS[5]); c5["n_sectors"] = 1; c5["n_rows"] = 4; c5["npads"] = gen.npads_linear(152, 66, 138)[::40][:4]
d5 = gen.generate(c5, frame=2)
g5 = gen.geometry(c5)
cl5, st5 = orc.run(d5, *g5[:4], npads=g5[4])
out["c5"] = [int(d5.shape[0]), st5["n_clusters"]]
e, se = orc.run(np.zeros(0, dtype=orc.DIGIT), 1, 1, 4, 4)
edge = orc.make_digits([(0, 0, 9), (3, 3, 9), (3, 0, 65535), (0, 3, 65535)])
ce, sedge = orc.run(edge, 1, 1, 4, 4)
out["edge"] = [se["n_clusters"], sedge["n_clusters"]]
out["dense"] = int(orc.dense_plane(d1, *g1[:4], 0, 7).astype(np.uint64).sum())
part, sp = orc.run(d1, *g1[:4], planes=(3, 9))
out["part"] = sp["n_clusters"]
# entropy coder oracle: round trip of config 1's clusters
buf, err, total = ec_oracle.encode(cl1, g1[0], g1[1])
back, derr = ec_oracle.decode(buf[:total])[:2]
out["ec"] = [int(err), int(total), int(derr), int(np.array_equal(back["qtot"], cl1["qtot"]))]
# front-end generator + filter oracle on a 3-row version of config 1
c1 = dict(gen.CONFIGS[1]); c1["n_rows"] = 3
d3 = gen.generate(c1)
g3 = gen.geometry(c1)
raw, ped4 = fe_gen.raw_from_digits(d3, *g3[:4], npads=g3[4], seed=1)
fd, fst = fe_oracle.run(raw, ped4, *g3[:4], npads=g3[4], zs_threshold=3)
out["fe"] = [int(raw.astype(np.uint64).sum() % (1 << 32)), fst["n_digits"]]
print(json.dumps(out))
