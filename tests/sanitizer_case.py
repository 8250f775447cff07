"""One small pass over every kernel family (C1-sized inputs), for `compute-sanitizer --tool <t> python tests/sanitizer_case.py`.
Not collected by pytest; results are checked only for having run (parity lives in the test files)."""
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import torch

import paper_1302_4000_b200 as pkg
from paper_1302_4000_b200 import workloads as wl


def main():
    pkg.load()
    for cfg, N in (("C1", None), ("C2", 300), ("C3", 200)):        # k-steps 3, 4 and 8; ragged tile edges
        ens = wl.make_config(cfg, N=N)
        x = torch.from_numpy(ens.coords).cuda()
        for eng in (pkg.ENGINE_I8TC, pkg.ENGINE_FFMA):
            pkg.clusco_crmsd_allpairs(x, engine=eng)
        pkg.clusco_crmsd_rowstats(x, 3.2)
        pkg.clusco_crmsd_allpairs_below(x, 3.2, 4096)
        pkg.clusco_center(x)
        pkg.clusco_drmsd_allpairs(x)
        pkg.clusco_cmo_allpairs(x, 8.0)
    ova = wl.make_config("C5", N=2000, chunk=2000)
    nat, co = torch.from_numpy(ova.native).cuda(), torch.from_numpy(ova.coords).cuda()
    pkg.clusco_crmsd_one_vs_all(nat, co)
    pkg.clusco_gdt_one_vs_all(nat, co[:64])
    torch.cuda.synchronize()
    print("sanitizer case ran")


if __name__ == "__main__":
    main()
