"""Writes the stored expected values under tests/golden/.  Calls ONLY oracle/ and the
seeded input generators (never the CUDA path).  Run from the repo root:

    python tests/golden/make_golden.py

c1_digest.json : sha256 of the oracle's codes / scales / int32 accumulators / bf16 output on
                 config 1 (BASELINE.json configs[0]) -- guards the oracle and the generator
                 against silent drift.
"""
import hashlib
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import oracle  # noqa: E402
from baseq_inputs import make_layer  # noqa: E402


def main():
    L = make_layer("c1", "linear")
    sp = L["spec"]
    fb = oracle.fused_bias(L["w_nibbles"], L["w_scale"], L["b"], L["layer_bias"])
    out = oracle.linear(L["x"], L["w_nibbles"], L["w_scale"], fb, sp.alpha, sp.gamma, None, L["b"])
    dig = {k: hashlib.sha256(out[k].tobytes()).hexdigest() for k in ("codes", "scales", "acc", "y")}
    dig["_written_by"] = "tests/golden/make_golden.py (oracle only)"
    with open(os.path.join(HERE, "c1_digest.json"), "w") as f:
        json.dump(dig, f, indent=1)
    print(dig)


if __name__ == "__main__":
    main()
