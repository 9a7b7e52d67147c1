"""Small invocations of every kernel of libsho.so, for compute-sanitizer (memcheck / racecheck / synccheck /
initcheck).  Not collected by pytest; run as

    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py [case ...]

Cases: cfg1, cfg2-small, cfg3-small, cfg4-small, cfg5-small (default: cfg1 cfg2-small cfg5-small).  Each case runs
project, add, the stored-projector project, the fused non-local action where the library has it, and the HOST-buffer
entry points, then prints a checksum.  No oracle comparison here: tests/test_gpu_parity.py does that; this script only
gives the sanitizer something to watch."""
import sys
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main(argv):
    import torch
    import paper_1905_00480_b200 as sho
    from paper_1905_00480_b200 import workloads

    names = argv or ["cfg1", "cfg2-small", "cfg5-small"]
    for name in names:
        k = int(name[3])
        w = workloads.make(k, size="small" if name.endswith("small") else "full")
        plan = sho.plan_for(w)
        psi_h = w.psi()
        if w.psi_dist == "zero":
            psi_h = workloads.Workload(**{**w.__dict__, "psi_dist": "normal"}).psi()
        psi = torch.from_numpy(psi_h).cuda()
        c = plan.project(psi)
        plan.add(c, psi)
        tb = plan.tables()
        c2 = plan.project_stored(tb, psi)
        torch.cuda.synchronize()
        tb.close()
        sums = [float(torch.abs(c).sum()), float(torch.abs(c2).sum()), float(torch.abs(psi).sum())]
        if hasattr(plan, "apply"):
            D = torch.from_numpy(w.dmatrix(plan.nsho)).cuda()
            plan.apply(D, psi)
            torch.cuda.synchronize()
            sums.append(float(torch.abs(psi).sum()))
        ch = np.zeros((w.natoms, w.nbands, plan.nsho), dtype=psi_h.dtype)
        plan.project_host(psi_h, ch)
        plan.add_host(ch, psi_h)
        sums.append(float(np.abs(psi_h).sum()))
        plan.close()
        print("%s ok: %s" % (name, " ".join("%.6e" % v for v in sums)))
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
