#!/usr/bin/env python
"""Writes tests/golden/recon.json: worked edge values (q-, q+) of PLM, PPM4, PPMX and WENOZ on the 9-point sequence of
SURVEY.md Appendix A.3, q = [1, 2, 4, 7, 8, 8.5, 3, 2.5, 2], cells 2..6.

Stand-alone: the vectorised numpy forms of make_appendix_c.py (the second, independently written implementation of the
readings DESIGN.md Q4, Q5, Q29, Q30), imports nothing from oracle/ or the CUDA package.  The sequence is treated as periodic by
those routines; cells 2..6 have their whole five-point stencil inside it, so the wrap never reaches them.

    python tests/golden/make_recon.py
"""
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import make_appendix_c as M     # noqa: E402

Q = [1, 2, 4, 7, 8, 8.5, 3, 2.5, 2]

if __name__ == "__main__":
    q = np.array(Q, dtype=float)
    out = {"source": "tests/golden/make_recon.py (numpy forms of make_appendix_c.py; DESIGN.md Q4, Q5, Q29, Q30)", "recon_q": Q}
    for name, fn in (("plm", M.plm), ("ppm4", M.ppm4), ("ppmx", M.ppmx), ("wenoz", M.wenoz)):
        qm, qp = fn(q)
        out[name] = {str(i): [float(qm[i]), float(qp[i])] for i in range(2, 7)}
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "recon.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out, indent=1))
