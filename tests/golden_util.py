"""Reader for tests/golden/*.txt (written by tests/golden/make_golden.py)."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_decode(name):
    rows, hist = [], None
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.startswith("# n_active_hist"):
                hist = [int(x) for x in line.split()[2:]]
            elif line.startswith("#") or not line.strip():
                continue
            else:
                p = line.split()
                rows.append((int(p[1]), int(p[2]), int(p[3]), float(p[4]), [int(x) for x in p[5:]]))
    return dict(
        len=np.array([r[0] for r in rows], np.int32),
        done=np.array([r[1] for r in rows], np.uint8),
        final_state=np.array([r[2] for r in rows], np.int32),
        sum_logprob=np.array([r[3] for r in rows], np.float64),
        tokens=np.array([r[4] for r in rows], np.int32),
        n_active_hist=np.array(hist, np.int32),
    )
