"""Writes tests/golden/full_size_oracle.txt: what the CPU oracle (and only the oracle) computes on the
full-size BASELINE.json configurations that are too slow to re-run inside the GPU test suite.

    python tests/golden/make_full_size_golden.py          (about 10 minutes on 8 cores)

cfg 4 (192^3 variable-coefficient diffusion, permuted rows): AMG-PCG to rtol 1e-8 from x0 = 0 -> iteration count,
recurrence residual, number of levels, rows / nonzeros per level.  The GPU test compares its own run with these
(iterations within +-2, identical level shapes) and checks the residual itself on the host in fp64.
"""
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_09001_b200 import inputs  # noqa: E402  (seeded generators only: no method arithmetic)


def main():
    out = []
    A = inputs.config_matrix(4, 192)
    b = inputs.config_rhs(4, A.n)
    t = time.time()
    o = oracle.Oracle(A.rowptr, A.col, A.val)
    ts = time.time() - t
    t = time.time()
    _, info = o.solve(b, 1e-8, 1000, 0, 1)
    tv = time.time() - t
    shapes = [o.level_info(l) for l in range(o.num_levels)]
    out.append("# written by tests/golden/make_full_size_golden.py (CPU oracle only); cfg 4 = BASELINE.json configs[3]")
    out.append(f"# oracle setup {ts:.0f} s, solve {tv:.0f} s on {os.cpu_count()} cores")
    out.append(f"cfg4_192 iterations {info.iterations}")
    out.append(f"cfg4_192 rel_residual {info.rel_residual:.17g}")
    out.append(f"cfg4_192 levels {o.num_levels}")
    out.append("cfg4_192 rows " + " ".join(str(r) for r, _ in shapes))
    out.append("cfg4_192 nnz " + " ".join(str(z) for _, z in shapes))
    o.close()
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "full_size_oracle.txt"), "w") as f:
        f.write("\n".join(out) + "\n")
    print("\n".join(out))


if __name__ == "__main__":
    main()
