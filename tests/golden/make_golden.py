"""Writes tests/golden/cfg1_oracle.json and tests/golden/next2_oracle.json: regression snapshots of the
CPU oracle on BASELINE.json configs[0] and on a crop of the contact-point + slot-feature config (the paper prints no renderer values to store instead --
SURVEY.md Sec.4).  Calls only oracle/ and the seeded input generator.

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import mso  # noqa: E402
from paper_2606_03877_b200 import synth  # noqa: E402

cfg = synth.CONFIGS["cfg1"]
sc = synth.make_scene(cfg)
cam = synth.make_cameras(cfg)[0]
rgb, alpha, _, st = mso.OracleScene(sc).render(cam, cfg.height, cfg.width, cfg.K)
hit = np.flatnonzero(alpha > 0)
pix = hit[:: max(1, len(hit) // 24)][:24].tolist() + [0, cfg.width * cfg.height - 1]
out = {"source": "oracle/mso.c via tests/golden/make_golden.py; BASELINE.json configs[0], seed 0",
       "n_intervals": st.n_intervals, "n_pairs": st.n_pairs, "pixels": pix,
       "rgb": rgb[pix].tolist(), "alpha": alpha[pix].tolist()}
with open(os.path.join(os.path.dirname(__file__), "cfg1_oracle.json"), "w") as f:
    json.dump(out, f, indent=1)
print("wrote", len(pix), "pixels")

# contact-point mode with Eq.7 slot features: a 96 x 54 crop of next2 with C_f = 8
from dataclasses import replace  # noqa: E402

cfg2 = synth.shrink(replace(synth.CONFIGS["next2"], c_f=8), 96, 54)
sc2 = synth.make_scene(cfg2)
cam2 = synth.make_cameras(cfg2)[0]
rgb2, alpha2, feat2, st2 = mso.OracleScene(sc2).render(cam2, 54, 96, 1)
pix2 = list(range(7, 96 * 54, 223))
out2 = {"source": "oracle/mso.c via tests/golden/make_golden.py; synth config next2 (seed 6) cropped to 96x54, C_f = 8, K = 1",
        "n_intervals": st2.n_intervals, "n_pairs": st2.n_pairs, "pixels": pix2,
        "rgb": rgb2[pix2].tolist(), "alpha": alpha2[pix2].tolist(), "feat": feat2[pix2].tolist()}
with open(os.path.join(os.path.dirname(__file__), "next2_oracle.json"), "w") as f:
    json.dump(out2, f, indent=1)
print("wrote", len(pix2), "pixels")
