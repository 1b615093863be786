"""Runs the paper's own instance grids (Figure 2 / Table 1 grid P:L317-333 and Figure 3 grid
P:L335) through meb_solve on cuda:0 and prints device times and the number of balls kept for phase 2.

    python -m paper_2605_31425_b200.paper_grid
"""
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_2605_31425_b200 as meb  # noqa: E402
import workloads  # noqa: E402


def main():
    rows=[]
    for d in (20,30,40,50):
        for m in (1000,5000,10000,50000,100000):
            C,R = workloads.paper_instance(m,d)
            dC,dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
            with meb.Context(m,d) as ctx:
                out={}
                for mode,name in ((0,'fp64'),(1,'mixed')):
                    for _ in range(3):
                        c,r,st = meb.meb_solve(ctx,dC,dR,1e-8,mode)
                    out[name]=(st['ms_total'],r,st['n_reduced'])
            rows.append((d,m,out['fp64'][0],out['mixed'][0],out['mixed'][2],out['mixed'][1]))
            print(d,m,"fp64 %.2f ms"%out['fp64'][0],"mixed %.2f ms"%out['mixed'][0],"kept",out['mixed'][2],"r %.8f"%out['mixed'][1], flush=True)
    for d in (100,500,1000,5000,10000):
        for m in (1000,5000):
            C,R = workloads.paper_instance(m,d)
            dC,dR = torch.from_numpy(C).cuda(), torch.from_numpy(R).cuda()
            with meb.Context(m,d) as ctx:
                out={}
                for mode,name in ((0,'fp64'),(1,'mixed')):
                    for _ in range(2):
                        c,r,st = meb.meb_solve(ctx,dC,dR,1e-8,mode,allow_not_converged=True)
                    out[name]=(st['ms_total'],r,st['n_reduced'],st['converged'])
            print(d,m,"fp64 %.2f ms"%out['fp64'][0],"mixed %.2f ms"%out['mixed'][0],"kept",out['mixed'][2],"conv",out['fp64'][3],out['mixed'][3],"r %.8f"%out['mixed'][1], flush=True)


if __name__ == "__main__":
    main()
