"""Writes tests/golden/setup_redraw_cases.json: global game indices whose fresh classic setup is
immobile at the first attempt and is redrawn (reading R5; p = 7*6*5*4*3*2 / (40*39*38*37*36*35)
= 1.8e-6 per side: the six front squares beside the lakes all hold Bombs / the Flag).
Calls only the oracle.  Run from the repository root:  python tests/golden/make_setup_redraw_cases.py"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import orc  # noqa: E402

SCAN = 2_000_000
cases = {"variant": 0, "seed": 0, "scanned_indices": SCAN,
         "citation": "DESIGN.md R5 (PAPER.md:234 is silent on immobile setups); found by oracle/orc.find_setup_redraws",
         "epoch0": orc.find_setup_redraws(0, 0, 0, 0, SCAN), "epoch1": orc.find_setup_redraws(0, 0, 1, 0, SCAN)}
with open(os.path.join(ROOT, "tests", "golden", "setup_redraw_cases.json"), "w") as f:
    json.dump(cases, f, indent=1)
print(cases)
