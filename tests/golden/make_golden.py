"""Writes tests/golden/cfg1_oracle.json: a regression snapshot of the CPU oracle on
BASELINE.json configs[0] (the paper prints no renderer values to store instead --
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
