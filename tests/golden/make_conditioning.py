#!/usr/bin/env python
"""Writes tests/golden/cfg{1,4}_conditioning.txt: how far the fp64 ORACLE's own 100-step trajectory of
every replica of config 1 / config 4 moves when its inputs are disturbed at the fp32 rounding level --
the conditioning of the 1e-4 A trajectory bar (reading S30).

Calls only oracle/ and the seeded generator (tier rule: no stored value comes from the CUDA path).
For each replica (256 of config 1, 4,096 of config 4; BASELINE.json:configs) it integrates 100 steps of
0.5 fs (O8) from the generator's state, then again from each disturbed state

  P1, P2, P3  every initial coordinate moved to the next fp32 value up or down, the signs drawn by
              numpy Generator(PCG64(k)), k = 1, 2, 3: three independent input errors of one fp32 ulp
              (the opposite sign pattern gives the same distance to 3 digits: the regime is linear);
  M           all four masses scaled by (1 + 2^-23): every acceleration off by one fp32 ulp,
              coherently, at every step (what a correctly rounded fp32 force would do at best);

and records the per-replica RMSD (A) between the disturbed and the undisturbed oracle at step 100.
No fp32 evaluation of F can be expected to track the fp64 trajectory of a replica closer than
these distances.  Config 4: about 22 minutes on 16 cores (five 100-step oracle runs of 227,857 atoms);
config 1: under a minute.

  python tests/golden/make_conditioning.py <config: 1 or 4> [n_replicas]
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle                                                    # noqa: E402
from paper_2412_18271_b200 import workloads as W                 # noqa: E402


def main():
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 4
    assert cfg in (1, 4)
    n_rep = int(sys.argv[2]) if len(sys.argv) > 2 else (4096 if cfg == 4 else 256)
    out_path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"cfg{cfg}_conditioning.txt")
    w = W.make_weights()
    wl = W.config4(n_replicas=n_rep) if cfg == 4 else W.config1(n_replicas=n_rep)
    off = wl.sys_offsets

    def rmsd(x, y):
        d2 = ((x - y) ** 2).sum(1)
        return np.array([np.sqrt(d2[off[s]:off[s + 1]].mean()) for s in range(len(off) - 1)])

    t0 = time.time()
    ref = oracle.step(wl.pos, wl.vel, wl.species, off, w, wl.dt_fs, 100)["pos"]
    print(f"baseline {time.time() - t0:.0f} s", flush=True)
    up, dn = np.nextafter(wl.pos, np.float32(np.inf)), np.nextafter(wl.pos, np.float32(-np.inf))
    cols = {}
    for k in (1, 2, 3):
        sgn = np.random.Generator(np.random.PCG64(k)).integers(0, 2, size=wl.pos.shape) * 2 - 1
        p = np.where(sgn > 0, up, dn).astype(np.float32)
        cols[f"P{k}"] = rmsd(oracle.step(p, wl.vel, wl.species, off, w, wl.dt_fs, 100)["pos"], ref)
        print(f"P{k} {time.time() - t0:.0f} s", flush=True)
    x = oracle.step(wl.pos, wl.vel, wl.species, off, w, wl.dt_fs, 100, masses=oracle.MASSES_AMU * (1.0 + 2.0 ** -23))["pos"]
    cols["M"] = rmsd(x, ref)
    print(f"M {time.time() - t0:.0f} s", flush=True)
    names = ("P1", "P2", "P3", "M")
    with open(out_path, "w") as f:
        f.write(f"# written by tests/golden/make_conditioning.py {cfg} (oracle only): per-replica RMSD (A) at step 100\n"
                "# between the fp64 oracle and the same oracle with inputs disturbed by one fp32 ulp\n"
                "# replica  n_atoms  P1  P2  P3  M\n")
        for s in range(len(off) - 1):
            f.write(f"{s} {off[s + 1] - off[s]} " + " ".join(f"{cols[k][s]:.4e}" for k in names) + "\n")
    worst = np.max([cols[k] for k in cols], axis=0)
    print("replicas whose worst disturbance exceeds 1e-4 A:", int((worst > 1e-4).sum()), "max", worst.max())


if __name__ == "__main__":
    main()
