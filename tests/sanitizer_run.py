"""Small driver for compute-sanitizer: a 2-group batch through every hot-path entry point.

    compute-sanitizer --tool memcheck|racecheck|initcheck|synccheck python tests/sanitizer_run.py [variant ...]

Variants: vl32 vl64 ctu32 ctu64 roe32 host32 (default: all).  No oracle, no assertions on values: the sanitizer's own
report is the result (profiles/r02_sanitizers.md); outputs are only checked for finiteness so that a kernel that was
skipped altogether cannot pass silently.
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_1804_03479_b200 import inputs, mhd  # noqa: E402

VARIANTS = {
    "vl32": dict(prec=mhd.FP32, scheme=mhd.VL, recon=mhd.PLM, g=3, riemann=mhd.HLLD),
    "vl64": dict(prec=mhd.FP64, scheme=mhd.VL, recon=mhd.PLM, g=3, riemann=mhd.HLLD),
    "ctu32": dict(prec=mhd.FP32, scheme=mhd.CTU, recon=mhd.PPM, g=4, riemann=mhd.HLLD),
    "ctu64": dict(prec=mhd.FP64, scheme=mhd.CTU, recon=mhd.PPM, g=4, riemann=mhd.HLLD),
    "roe32": dict(prec=mhd.FP32, scheme=mhd.VL, recon=mhd.PLM, g=3, riemann=mhd.ROE),
    "host32": dict(prec=mhd.FP32, scheme=mhd.VL, recon=mhd.PLM, g=3, riemann=mhd.HLLD, host=True),
}


def run(name, prec, scheme, recon, g, riemann, host=False, G=2, N=16):
    npdt = np.float32 if prec == mhd.FP32 else np.float64
    U, B, dh = inputs.config2_batch(G, N=N, g=g, dtype=npdt)
    s = mhd.Solver(mhd.make_config(N=N, g=g, prec=prec, scheme=scheme, recon=recon, riemann=riemann, max_groups=G))
    if host:
        tdt = torch.float32 if prec == mhd.FP32 else torch.float64
        hU, hB = torch.from_numpy(U).pin_memory(), torch.from_numpy(B).pin_memory()
        ho = {k: torch.empty((G, n), dtype=tdt).pin_memory() for k, n in
              (("U", s.n_U_out), ("B", s.n_B_out), ("flux", s.n_flux), ("emf", s.n_emf))}
        dtn, _ = s.advance_host_dt(hU, hB, ho["U"], ho["B"], ho["flux"], ho["emf"], G, 2e-3, dh, 1, 2, 0.3)
        outs = {k: v.numpy() for k, v in ho.items()}
    else:
        dU, dB = torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda()
        dt0, _ = s.dt_reduce(dU, dB, G, g, dh, 0.3)
        out = s.alloc_outputs(G)
        dtn, _ = s.advance_dt(dU, dB, out["U"], out["B"], out["flux"], out["emf"], G, dt0, dh, 0.3)
        s.advance(dU, dB, out["U"], out["B"], None, None, G, dt0, dh)
        torch.cuda.synchronize()
        outs = {k: v.cpu().numpy() for k, v in out.items()}
    for k, v in outs.items():
        assert np.isfinite(v).all(), (name, k)
    assert np.isfinite(dtn) and dtn > 0
    nl = s.launch_count()
    s.destroy()
    print(f"{name}: ok, {nl} launches", flush=True)


if __name__ == "__main__":
    names = sys.argv[1:] or list(VARIANTS)
    for nm in names:
        run(nm, **VARIANTS[nm])
