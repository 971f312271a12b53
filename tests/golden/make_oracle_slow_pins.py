"""Writes tests/golden/oracle_slow_pins.json: the values of the two long oracle pins of tests/test_oracle_hydro.py
(PAPER.md:299 at N = 1024) with the SHA-256 fingerprint of the files they depend on (oracle sources, the
oracle's build flags, the test module).  Calls only the test module's own functions, which call only oracle/ -- nothing
from the CUDA path.  Run after any change of oracle/ or of tests/test_oracle_hydro.py:

    python tests/golden/make_oracle_slow_pins.py        # ~6 minutes on 8 cores
"""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))                       # tests/
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))      # repository root (oracle/)

import test_oracle_hydro as T  # noqa: E402

if __name__ == "__main__":
    values = {"sound_wave_error_1024": T._sound_wave_error(1024), "strong_shock_rel_error": T._strong_shock_rel_error()}
    out = {"fingerprint": T._oracle_fingerprint(),
           "what": "values computed by the CPU oracle alone; tests/test_oracle_hydro.py compares them with the paper's "
                   "printed numbers (PAPER.md:299, 313) and recomputes them when the fingerprint no longer matches",
           "values": values}
    with open(T.SLOW_PINS, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print(json.dumps(out, indent=1))
