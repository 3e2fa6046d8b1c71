"""Writes tests/golden/oracle_water64.txt: oracle energy and a few force components for the seeded 64-water box
(BASELINE.json configs[0]) -- a regression pin for oracle/ itself.  Calls only oracle/ and the input generators.
The paper prints no value for this path (SURVEY.md 8(c) C3 last row), so these numbers are the oracle's own."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import nnp_oracle as orc              # noqa: E402
from paper_2405_01491_b200 import inputs          # noqa: E402

consts = inputs.ani2x_constants()
params = inputs.make_weights(inputs.SEED0, 1, last_layer_scale=inputs.FORCE_SCALE_WATER, bias_std=0.05)
om = orc.OracleModel(consts, inputs.WIDTHS, params, 1)
sp, xyz, box = inputs.water_box(64, 12.42)
r = orc.energy_forces(om, sp, xyz, box, want_aev=True)
out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_water64.txt")
with open(out, "w") as f:
    f.write("# oracle/nnp_oracle.c on inputs.water_box(64, 12.42), weights seed %d scale %g bias_std 0.05\n" % (inputs.SEED0, inputs.FORCE_SCALE_WATER))
    f.write("E %.12e\n" % r["E"][0])
    for i in (0, 1, 2, 95, 191):
        f.write("F %d %.12e %.12e %.12e\n" % (i, *r["F"][i]))
    f.write("AEVSUM %.12e\n" % r["aev"].sum())
    f.write("AEVNNZ %d\n" % int((r["aev"] != 0).sum()))
print(open(out).read())
