#!/usr/bin/env python
"""Writes tests/golden/cfg3_traj10.npz: BASELINE.json config 3 (64^3 cells, 1e6 beam electrons) after 10 full PIC steps
of the fp64 CPU oracle (deposit -> push_sources -> field_step -> push_particles; PAPER.md:85 section 2, :231 section 2.4).

It calls ONLY `oracle/` and the seeded input generator `paper_2209_07944_b200.workloads` (which holds none of the
method's arithmetic); nothing here loads or runs the CUDA library.  The GPU test that reads the file is
tests/test_gpu_fullsize.py::test_config3_closed_loop_10_steps_golden (north_star: "particle positions must match within
1e-5 relative after 10 steps"; "config 3: full closed-loop oracle for the first 10 steps").

Cost: 10 steps x 6.87e10 source-observation pairs in fp64; about two hours on 8 host cores (the header of the file records
the cores and the wall time of the run that wrote it).  `--ckpt FILE` saves the state after every step and resumes from it.

Stored (the whole state would be 60 MB; a 1e6-particle trajectory depends on every other particle only through E and B,
so a seeded subset of trajectories plus population sums pins the run):
  sub_idx [32768]            seeded subset of particle numbers (numpy default_rng([seed, 10]).choice)
  sub_x..sub_uz [32768] f64  their state after step 9's push (r^10 in grid units, u^{9+1/2})
  alive_bits                 np.packbits of the alive flag of ALL particles after step 9
  sum_xyz [3], sum_u [3] f64 sums over all alive particles
  obs [4096+15]              wl.sample_obs(64, 4096, seed): cells where fields and sources of step 9 are kept
  E9, B9 [3][nobs] f64       fields of step 9 at those cells;  S9 [4][nobs] f64 deposited rho, J of step 9
  E9_norm, B9_norm           L2 norms over ALL cells (the denominators of the field tolerances)
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

STEPS = 10
NSUB = 32768
NOBS = 4096


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(HERE, "cfg3_traj10.npz"))
    ap.add_argument("--ckpt", default=None, help="checkpoint file: state saved after every step, resumed if present")
    ap.add_argument("--threads", type=int, default=0)
    ap.add_argument("--private-lib", default=None,
                    help="copy libjefi_oracle.so to this path and load the copy (so that the oracle can be rebuilt meanwhile)")
    args = ap.parse_args()

    import oracle
    from oracle import jefi_oracle as jo
    from paper_2209_07944_b200 import workloads as wl

    if args.private_lib:
        import shutil

        shutil.copy(oracle.build_oracle(), args.private_lib)
        jo._LIB = args.private_lib
        jo.build_oracle = lambda force=False: args.private_lib
    if args.threads:
        oracle.set_num_threads(args.threads)
    w = wl.WORKLOADS[3]
    cfg = oracle.OracleConfig(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt)
    assert cfg.H == w.H
    part = wl.particles(3)
    P = part["x"].shape[0]
    po = {k: v.astype(np.float64) for k, v in part.items() if k != "alive"}
    po["alive"] = part["alive"].copy()
    orc = oracle.OracleJefi(cfg)
    done, wall = 0, 0.0
    if args.ckpt and os.path.exists(args.ckpt):
        ck = np.load(args.ckpt)
        done, wall = int(ck["done"]), float(ck["wall"])
        for k in po:
            po[k] = ck["p_" + k].copy()
        orc.ring[:done] = ck["ring"]
        orc.n = done - 1
        print(f"resumed after step {done - 1} ({wall:.0f} s so far)", flush=True)
    S = E = B = None
    for s in range(done, STEPS):
        t0 = time.perf_counter()
        S, E, B = orc.pic_step(po)
        wall += time.perf_counter() - t0
        print(f"step {s}: {time.perf_counter() - t0:.0f} s, alive {int(po['alive'].sum())}, |E| {np.linalg.norm(E):.6e}", flush=True)
        if args.ckpt and s < STEPS - 1:
            np.savez(args.ckpt + ".tmp.npz", done=s + 1, wall=wall, ring=orc.ring[:s + 1], **{"p_" + k: v for k, v in po.items()})
            os.replace(args.ckpt + ".tmp.npz", args.ckpt)
    assert S is not None, "nothing left to do (checkpoint already at the last step): delete it to rerun"
    sub = np.sort(np.random.default_rng([w.seed, 10]).choice(P, NSUB, replace=False)).astype(np.int64)
    obs = wl.sample_obs(w.n, NOBS, w.seed)
    al = po["alive"] == 1
    header = (f"cfg3 (64^3, dx=5e-5, dt=dx/2c, H={cfg.H}, {P} macro-electrons, seed {w.seed}) after {STEPS} oracle PIC steps; "
              f"written by tests/golden/make_cfg3_traj10.py calling only oracle/ (fp64, {oracle.num_threads()} host threads, "
              f"{wall:.0f} s of wall time in pic_step)")
    np.savez_compressed(
        args.out, header=np.array(header), sub_idx=sub,
        **{"sub_" + k: po[k][sub] for k in ("x", "y", "z", "ux", "uy", "uz")},
        alive_bits=np.packbits(po["alive"]), n_alive=np.int64(al.sum()),
        sum_xyz=np.array([po[k][al].sum() for k in "xyz"]), sum_u=np.array([po[k][al].sum() for k in ("ux", "uy", "uz")]),
        obs=obs, E9=E[:, obs], B9=B[:, obs], S9=S[:, obs], E9_norm=np.linalg.norm(E), B9_norm=np.linalg.norm(B),
        E9_absmax=np.abs(E).max(), B9_absmax=np.abs(B).max())
    print(header)
    print("wrote", args.out, os.path.getsize(args.out), "bytes")


if __name__ == "__main__":
    main()
