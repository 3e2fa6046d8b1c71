"""Writes tests/golden/force_scale.md: the oracle's RMS force and atomic-energy spread on the 64-water box for
the seeded Xavier weights at last-layer scale 1 (reading B7).  Calls only oracle/ and the input generators."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import nnp_oracle as orc              # noqa: E402
from paper_2405_01491_b200 import inputs          # noqa: E402

consts = inputs.ani2x_constants()
om = orc.OracleModel(consts, inputs.WIDTHS, inputs.make_weights(inputs.SEED0, 1), 1)
sp, xyz, box = inputs.water_box(64, 12.42)
r = orc.energy_forces(om, sp, xyz, box, want_e_atom=True)
frms = float(np.sqrt((r["F"] ** 2).sum(1).mean()))
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "force_scale.md"), "w") as f:
    f.write("# Force scale of the seeded random-weight model (reading B7)\n\n")
    f.write("Written by `tests/golden/derive_force_scale.py` (oracle only).  64-water box, seed %d, last-layer scale 1:\n\n" % inputs.SEED0)
    f.write("- RMS |F| = %.4f kcal/mol/A\n- std of atomic energies = %.4f kcal/mol\n- E = %.6f kcal/mol\n\n" % (frms, r["e_atom"].std(), r["E"][0]))
    f.write("`inputs.FORCE_SCALE_WATER = 66` brings RMS |F| to about %.1f kcal/mol/A (liquid-water-like) for the parity tests;\n" % (66 * frms))
    f.write("`inputs.FORCE_SCALE_MD = 2` (RMS |F| about %.2f) is used for MD workloads, see DESIGN.md \"Input recipe\".\n" % (2 * frms))
print(frms)
