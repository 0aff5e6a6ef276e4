"""FP32 control experiment (reading R14b) -- run on the GPU box:

    python -m paper_1804_03479_b200.build --ieee32 && python tests/fp32_controls.py > gpurun_out/fp32_controls.md

For the FP32 parity cases it prints, per field, the error against the FP64 oracle (same FP32-rounded inputs, the oracle's
dt sequence, emf_tie = 1e-5 on every side) of three FP32 implementations:
  oracle-FP32   the oracle source instantiated in single precision, every operation IEEE-rounded (oracle/mhd_oracle_f32.cpp)
  GPU           the CUDA path as shipped (SFU reciprocal / sqrt approximations, batched reciprocals)
  GPU-IEEE      the same kernels built with -DMHD_IEEE32 (IEEE-rounded FP32 division and square root)
The first column is the error inherent to running the plain algorithm in single precision: the gate of the -m gpu tests is
max(1e-4, 2 x that) per field (tests/parity_cases.fp32_gate).  The GPU-IEEE leg runs in a child process (MHD_LIBPATH).
"""
import json
import os
import subprocess
import sys
import tempfile

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.join(ROOT, "tests")):
    if p not in sys.path:
        sys.path.insert(0, p)

from paper_1804_03479_b200 import inputs  # noqa: E402
import gpu_util as GU  # noqa: E402
import parity_cases as PC  # noqa: E402

N = 16
CASES = {  # name: (scheme, recon, g, limvar)
    "config2_24boxes_10steps_VL+PLM": (0, 0, 3, 0),
    "config3_64cubed_10steps_CTU+PPM": (1, 1, 4, 1),
    "config3_256cubed_1step_26groups_CTU+PPM": (1, 1, 4, 1),
    "config5_first512of1024cubed_1step_VL+PLM": (0, 0, 3, 0),
    "config5_first512of1024cubed_1step_CTU+PPM": (1, 1, 4, 1),
}
SAMPLE5 = list(range(3, 512, 32))


def initial(case):
    if case.startswith("config2"):
        return PC.config2_boxes(24, N, prec=0)
    if case.startswith("config3_64"):
        return PC.config3_grid(64, prec=0)
    if case.startswith("config3_256"):
        g = CASES[case][2]
        (U, bx, by, bz), dh = PC.config3_grid(256, prec=0)
        Ui, Bi = inputs.pack_groups(U, bx, by, bz, N, g, np.float32)
        sample = list(range(7, 4096, 173)) + [4096 // 2 + 8 * 16 + 8, 4096 // 2 - 8 * 16 - 8 - 1]
        return (Ui[sample], Bi[sample]), dh
    g = CASES[case][2]
    Ui, Bi, dh = inputs.abc_groups(1024, 0, 512, N, g, dtype=np.float32)
    return (Ui, Bi), dh


def run(case, adv, dts, dtype, host_solver=None):
    """-> dict of arrays: the final state (multi-step cases) or the outputs of the one step"""
    scheme, recon, g, limvar = CASES[case]
    init, dh = initial(case)
    if case.startswith("config2"):
        boxes, out = PC.run_boxes(adv, init, dts, dh, N, g, dtype)
        res = {f"box{q}_{i}": np.asarray(a, dtype=np.float64) for q, b in enumerate(boxes) for i, a in enumerate(b)}
        res.update({"out_" + k: np.asarray(v, dtype=np.float64) for k, v in out.items() if k in ("U", "B", "flux", "emf")})
        return res
    if case.startswith("config3_64"):
        state, out = PC.run_grid(adv, init, dts, dh, N, g, dtype)
        res = {f"s{i}": np.asarray(a, dtype=np.float64) for i, a in enumerate(state)}
        res.update({"out_" + k: np.asarray(v, dtype=np.float64) for k, v in out.items() if k in ("U", "B", "flux", "emf")})
        return res
    Ui, Bi = init
    if case.startswith("config5") and host_solver is not None:
        out = host_solver(Ui, Bi, dts[0], dh)
    else:
        out = adv(Ui.astype(dtype), Bi.astype(dtype), dts[0], dh)
    if case.startswith("config5"):
        out = {k: np.asarray(v)[SAMPLE5] for k, v in out.items() if k in ("U", "B", "flux", "emf")}
    return {"out_" + k: np.asarray(v, dtype=np.float64) for k, v in out.items() if k in ("U", "B", "flux", "emf")}


def errors(case, res, ref):
    e = {}
    if case.startswith("config2"):
        G = 24
        a = [tuple(res[f"box{q}_{i}"] for i in range(4)) for q in range(G)]
        b = [tuple(ref[f"box{q}_{i}"] for i in range(4)) for q in range(G)]
        e.update(PC.boxes_errors(a, b))
    elif case.startswith("config3_64"):
        e.update(PC.grid_errors(tuple(res[f"s{i}"] for i in range(4)), tuple(ref[f"s{i}"] for i in range(4))))
    o = GU.field_errors({k[4:]: v for k, v in res.items() if k.startswith("out_")}, {k[4:]: v for k, v in ref.items() if k.startswith("out_")}, N)
    if case.startswith(("config2", "config3_64")):
        o = {k: v for k, v in o.items() if k.startswith(("flux", "emf"))}      # the state itself is compared above
    e.update(o)
    return e


def gpu_adv(case):
    scheme, recon, g, limvar = CASES[case]
    G = 512 if case.startswith("config5") else 64
    return GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, riemann=1, limvar=limvar, prec=0, max_groups=G)


def gpu_host_adv(runner):
    """config 5: through mhd_advance_host, 32-group chunks on 4 streams (BASELINE.json configs[4])"""
    import torch

    def adv(Ui, Bi, dt, dh):
        s = runner.solver
        G = Ui.shape[0]
        hU, hB = torch.from_numpy(np.ascontiguousarray(Ui)).pin_memory(), torch.from_numpy(np.ascontiguousarray(Bi)).pin_memory()
        ho = {k: torch.empty((G, n), dtype=torch.float32).pin_memory() for k, n in
              (("U", s.n_U_out), ("B", s.n_B_out), ("flux", s.n_flux), ("emf", s.n_emf))}
        s.advance_host(hU, hB, ho["U"], ho["B"], ho["flux"], ho["emf"], G, dt, dh, 32, 4)
        return {k: v.numpy().copy() for k, v in ho.items()}
    return adv


def child(case, dts, path):
    runner = gpu_adv(case)
    res = run(case, runner, dts, np.float32, host_solver=gpu_host_adv(runner) if case.startswith("config5") else None)
    np.savez(path, **res)


def main():
    from oracle import mhdref
    mhdref.build()
    from paper_1804_03479_b200 import build as B
    ieee = B.build_ieee32()
    print("# FP32 control experiment (tests/fp32_controls.py): err_f = max|x - oracle64| / max|oracle64| per field (R14)\n")
    print("Command: `python -m paper_1804_03479_b200.build --ieee32 && python tests/fp32_controls.py`\n")
    for case, (scheme, recon, g, limvar) in CASES.items():
        cfg = mhdref.make_config(N=N, g=g, scheme=scheme, recon=recon, riemann=1, limvar=limvar, emf_tie=PC.EMF_TIE[0])
        adv64 = lambda Ui, Bi, dt, dh_: mhdref.advance(cfg, Ui, Bi, dt, dh_)
        adv32 = lambda Ui, Bi, dt, dh_: mhdref.advance32(cfg, Ui, Bi, dt, dh_)
        init, dh = initial(case)
        # the FP64 oracle's own dt sequence
        if case.startswith("config2"):
            dts = PC.run_boxes_oracle(mhdref, cfg, init, dh, N, g)[0]
        elif case.startswith("config3_64"):
            dts = PC.run_grid_oracle(mhdref, adv64, init, dh, N, g)[0]
        else:
            Ui, Bi = init
            dts = [mhdref.dt_reduce(cfg, Ui.astype(np.float64), Bi.astype(np.float64), g, dh, 0.3)[0]]
        if case.startswith("config5"):
            # the oracle on the sampled groups only (groups are independent given their ghost zones)
            samp = lambda f: (lambda Ui, Bi, dt, dh_: {k: _expand(v, SAMPLE5, Ui.shape[0]) for k, v in
                                                         f(Ui[SAMPLE5], Bi[SAMPLE5], dt, dh_).items() if k in ("U", "B", "flux", "emf")})
            ref = run(case, samp(adv64), dts, np.float64)
            r32 = run(case, samp(adv32), dts, np.float32)
        else:
            ref = run(case, adv64, dts, np.float64)
            r32 = run(case, adv32, dts, np.float32)
        runner = gpu_adv(case)
        rgpu = run(case, runner, dts, np.float32, host_solver=gpu_host_adv(runner) if case.startswith("config5") else None)
        with tempfile.TemporaryDirectory() as td:
            path = os.path.join(td, "ieee.npz")
            env = dict(os.environ, MHD_LIBPATH=ieee)
            subprocess.check_call([sys.executable, os.path.abspath(__file__), "--child", case, json.dumps(dts), path], env=env)
            rie = dict(np.load(path))
        e32, eg, ei = errors(case, r32, ref), errors(case, rgpu, ref), errors(case, rie, ref)
        gate = PC.fp32_gate(e32)
        print(f"## {case}  (dt[0] = {dts[0]:.4e}, {len(dts)} step(s))\n")
        print("| field | oracle-FP32 | GPU | GPU-IEEE | gate = max(1e-4, 2 x oracle-FP32) | GPU / gate |")
        print("|---|---|---|---|---|---|")
        for k in e32:
            print(f"| {k} | {e32[k]:.2e} | {eg[k]:.2e} | {ei[k]:.2e} | {gate[k]:.2e} | {eg[k] / gate[k]:.2f} |")
        print(flush=True)


def _expand(v, sample, G):
    out = np.zeros((G,) + np.asarray(v).shape[1:], dtype=np.asarray(v).dtype)
    out[sample] = v
    return out


if __name__ == "__main__":
    if len(sys.argv) > 1 and sys.argv[1] == "--child":
        child(sys.argv[2], json.loads(sys.argv[3]), sys.argv[4])
    else:
        main()
