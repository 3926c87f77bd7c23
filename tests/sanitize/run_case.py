"""One small evaluation per kernel family, for compute-sanitizer runs (profiles/r2_sanitizer_*.txt name the commands):

    compute-sanitizer --tool racecheck python tests/sanitize/run_case.py 8
    compute-sanitizer --tool memcheck  python tests/sanitize/run_case.py 14

The batch is chosen so that every persistent CTA loops over at least two teams (prefetch into the live W area, re-use
of the shared-memory / scratch regions); the result is compared with the plain kernel of the same library."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))

import numpy as np
import torch

from paper_2501_00675_b200 import api

BATCH = {4: 5000, 8: 9600, 10: 2500, 11: 1300, 12: 700, 13: 310, 14: 310, 16: 300}


def main():
    n = int(sys.argv[1])
    nsp = int(sys.argv[2]) if len(sys.argv) > 2 else 1
    B = BATCH.get(n, 600)
    rng = np.random.default_rng(n)
    G = torch.from_numpy(rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)).cuda()
    G2 = torch.from_numpy(rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)).cuda() if nsp == 2 else G
    out = torch.empty(B, dtype=torch.float64, device="cuda")
    with api.Context() as c:
        c.eval_connected(G, G2, out, U=1.3)
        torch.cuda.synchronize()
        name = c.last_kernel_name()
        K = 16
        ref = torch.empty(K, dtype=torch.float64, device="cuda")
        c.force_generic(True)
        c.eval_connected(G[-K:].contiguous(), G2[-K:].contiguous() if nsp == 2 else G[-K:].contiguous(), ref, U=1.3)
        torch.cuda.synchronize()
    err = ((out[-K:] - ref).abs() / ref.abs()).max().item()
    print(f"n={n} nsp={nsp} batch={B} kernel={name} max rel diff vs plain kernel {err:.2e}")
    assert err < 1e-9


if __name__ == "__main__":
    main()
