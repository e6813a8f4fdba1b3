"""Writes tests/golden/oracle_cfg*.json: oracle Omega values on seeded sub-samples of the large BASELINE configs.

Calls ONLY oracle/ (never the CUDA path).  The GPU parity tests at full size (configs 3-5) compare against
these stored values so that the GPU box does not spend minutes of host time re-deriving them; the samples are
whole (q, h) columns for configs 3-4 (so the argmin check is meaningful) and strided Delta subsets of columns
for config 5.  Floats are stored with repr() (exact round trip).

    python tests/golden/make_golden.py [3 4 5]
"""
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import fe_oracle as O                     # noqa: E402
from paper_1412_8754_b200 import workloads as W      # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))

PLAN = {            # cfg: (number of (q,h) columns, Delta indices per column or None = all)
    3: (12, None),
    4: (4, None),
    5: (3, 24),
}


def delta_subset(nd, n):
    if n is None or n >= nd:
        return list(range(nd))
    idx = sorted(set(np.linspace(0, nd - 1, n).round().astype(int).tolist()))
    return idx


def main(cfgs):
    for c in cfgs:
        w = W.config(c)
        ncol, nsub = PLAN[c]
        cols = W.sample_columns(w, ncol, c)
        ids = delta_subset(w.nd, nsub)
        out = dict(config=c, workload=w.name, N=w.N, params=w.params, oracle="oracle/fe_oracle.c feo_omega_column",
                   generated_by="tests/golden/make_golden.py", runs=[])
        for T in w.T:
            t0 = time.time()
            entries = []
            for (iq, ih) in cols:
                om = O.omega_column(w.params, w.N, T, w.q[iq], w.h[ih], w.delta[ids])
                entries.append(dict(iq=iq, ih=ih, q=[repr(float(x)) for x in w.q[iq]], h=repr(float(w.h[ih])),
                                    id=ids, omega=[repr(float(x)) for x in om]))
                print(f"cfg{c} T={T} col ({iq},{ih}) done, {time.time() - t0:.1f}s", flush=True)
            out["runs"].append(dict(T=T, columns=entries))
        with open(os.path.join(HERE, f"oracle_cfg{c}.json"), "w") as f:
            json.dump(out, f, indent=0)
        print("wrote", f.name, flush=True)


if __name__ == "__main__":
    main([int(x) for x in sys.argv[1:]] or [3, 4, 5])
