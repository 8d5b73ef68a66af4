"""Writes the `value` fields of closed_forms.json from the hand-derived formulas stated in its
`_about` (pure `math`; calls neither oracle/ nor the CUDA path).  Run: python tests/golden/make_closed_forms.py"""
import json
import math
import os

path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "closed_forms.json")
d = json.load(open(path))
sad, sdd, du = d["sad"], d["sdd"], d["pitch"]
for c in d["sphere"]["cases"]:
    b = sad * math.sin(math.atan(c["m"] * du / sdd))
    c["value"] = 2.0 * d["sphere"]["rho"] * math.sqrt(d["sphere"]["r"] ** 2 - b * b)
for c in d["gauss"]["cases"]:
    b = sad * math.sin(math.atan(c["m"] * du / sdd))
    s = d["gauss"]["sigma"]
    c["value"] = d["gauss"]["a"] * s * math.sqrt(2 * math.pi) * math.exp(-b * b / (2 * s * s))
json.dump(d, open(path, "w"), indent=2)
print(json.dumps(d, indent=2))
