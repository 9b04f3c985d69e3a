"""The paper's beamlet-parameter search (Fig. 8-9) on the GPU.

`airy_sweep` is the batched C-ABI call gbd_airy_sweep (one grouped field-sum launch for all runs, no
synchronisation).  `airy_sweep_per_run` drives the same search run by run through the three basic
calls -- a1 lattice, a2 parameters, a3+a4 field, a 1x1 on-axis evaluation for the peak normalisation,
and the Airy figure of merit -- and is kept as the cross-check of the batched call.
"""
from __future__ import annotations

import torch

from . import gbd


def airy_sweep(runs, abcd, l0, detector, lambda_fnum, precision=gbd.PRECISION_FP64,
               algo=gbd.ALGO_DIRECT, device="cuda:0"):
    """Batched search (gbd_airy_sweep).  Returns a (len(runs), 10) CPU tensor."""
    return gbd.airy_sweep(runs, abcd, l0, detector, lambda_fnum, precision=precision, algo=algo,
                          device=device).cpu()


def airy_sweep_per_run(runs, abcd, l0, detector, lambda_fnum, precision=gbd.PRECISION_FP64,
                       algo=gbd.ALGO_DIRECT, device="cuda:0"):
    """runs: iterable of (n_across, pupil_diameter, overlap_factor, wavelength).
    abcd: shared 4x4 (16 doubles) of the optics; l0 its axial path; detector: dict; lambda_fnum = lambda F#.
    Returns a (len(runs), 10) CPU tensor: the 9 values of gbd_psf_metrics and the beamlet count."""
    device = torch.device(device)
    runs = list(runs)
    d_abcd = torch.as_tensor(abcd, dtype=torch.float64, device=device).reshape(16)
    out = torch.zeros((len(runs), 10), dtype=torch.float64, device=device)
    dtype = torch.complex128 if precision == gbd.PRECISION_FP64 else torch.complex64
    field = torch.empty((detector["n_v"], detector["n_u"]), dtype=dtype, device=device)
    e0 = torch.empty((1, 1), dtype=torch.complex128, device=device)
    det0 = dict(detector, n_u=1, n_v=1)
    mws = torch.empty(max(256, gbd.load_library().gbd_psf_metrics_workspace_bytes(
        gbd.C.byref(gbd.Detector.from_dict(detector)))), dtype=torch.uint8, device=device)
    keep = []
    for i, (n_across, diameter, of, lam) in enumerate(runs):
        b = gbd.beamlets_create(n_across, diameter, of, lam, device=device)
        gbd.propagate_q(b, 1, d_abcd, l0)
        gbd.eval_field(b, detector, precision=precision, algo=algo, out=field)
        gbd.eval_field(b, det0, out=e0)
        gbd.psf_metrics(field, detector, lambda_fnum, e0, out=out[i, :9], workspace=mws)
        out[i, 9] = float(b.n)
        keep.append(b)                      # keep workspaces alive until the stream has drained
    res = out.cpu()
    del keep
    return res


def runtime_vs_beamlets(n_list=range(11, 102, 10), overlap_factor=1.5, det_n=256, device="cuda:0", reps=5):
    """Shape of the paper's runtime experiment (Fig. 7: one 256 x 256 px PSF against the number of
    beamlets across the pupil), on the synthetic ideal-lens optics of BASELINE.json configs[2].
    Returns rows (n_across, beamlets, {algo: ms}) -- device time of gbd_eval_field, best of `reps`."""
    lam, diam, f = 0.6328e-3, 25.4, 100.0
    half = 8.0 * lam * f / diam
    det = dict(n_u=det_n, n_v=det_n, du=2 * half / det_n, dv=2 * half / det_n, origin=[0.0, 0.0, 0.0],
               e_u=[1.0, 0.0, 0.0], e_v=[0.0, 1.0, 0.0])
    abcd = [0, 0, f, 0, 0, 0, 0, f, -1 / f, 0, 1, 0, 0, -1 / f, 0, 1]
    rows = []
    for n in n_list:
        b = gbd.beamlets_create(n, diam, overlap_factor, lam, device=device)
        gbd.propagate_q(b, 1, abcd, f)
        out = {}
        for name, algo in (("direct", gbd.ALGO_DIRECT), ("recurrence", gbd.ALGO_RECURRENCE),
                           ("separable", gbd.ALGO_SEPARABLE)):
            fld = gbd.eval_field(b, det, algo=algo)
            torch.cuda.synchronize()
            best = None
            for _ in range(reps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                gbd.eval_field(b, det, algo=algo, out=fld, workspace=b._ws)
                e1.record()
                torch.cuda.synchronize()
                t = e0.elapsed_time(e1)
                best = t if best is None else min(best, t)
            out[name] = best
        rows.append((n, b.n, out))
    return rows


if __name__ == "__main__":
    print("| beamlets across | beamlets | terms | direct ms | recurrence ms | separable ms |")
    print("|---|---|---|---|---|---|")
    for n, nb, t in runtime_vs_beamlets():
        print(f"| {n} | {nb} | {nb * 65536:.3g} | {t['direct']:.4f} | {t['recurrence']:.4f} | {t['separable']:.4f} |")
