"""Measured parity of the CUDA path against the oracle, as a table (the gates themselves are asserted in
tests/test_gpu_parity.py; this prints how far inside them the path sits).

    python tests/parity_report.py > profiles/r1_parity.md        # needs a B200; ~2 minutes

Every row: seeded synthetic counts of the named config (synthgen), reconstructed through the C ABI and by the
oracle (oracle.recon, double precision) on the same arrays; rel-L2 per slice (max over the slices compared) and
max-abs over the slices divided by max |oracle| (reading Q14).
"""
from __future__ import annotations

import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle as orc  # noqa: E402
import paper_2209_08450_b200 as tcp  # noqa: E402
import synthgen as sg  # noqa: E402


def rl2(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def case(label, w, rows, dtype, method="grid", alg="fourier", pad="zero", tcfft=0, gpu_inputs=False, cut=None):
    """cut = (lo, hi): only detector columns lo..hi are passed on (a width that is not a power of two, tcp_create_det)."""
    nz = len(rows)
    lo, hi = cut if cut else (0, w.n)
    ndet, center = hi - lo, w.center - lo
    if gpu_inputs:
        raw_d, ff, df = sg.make_counts_torch(w, rows, device="cuda")
        flat_d = torch.empty((nz, w.n), dtype=torch.float32, device="cuda")
        dark_d = torch.empty_like(flat_d)
        tcp.tcp_mean_frames_u16(ff.contiguous(), flat_d)
        tcp.tcp_mean_frames_u16(df.contiguous(), dark_d)
        raw_d = raw_d.contiguous()
        theta_d = torch.from_numpy(w.theta).cuda()
    else:
        raw, _ = sg.make_counts(w, rows)
        flat, dark, _, _ = sg.make_flat_dark(w, rows)
        raw_d = torch.from_numpy(raw.view(np.int16)).cuda().view(torch.uint16)
        flat_d, dark_d, theta_d = torch.from_numpy(flat).cuda(), torch.from_numpy(dark).cuda(), torch.from_numpy(w.theta).cuda()
    if cut:
        raw_d = raw_d[:, :, lo:hi].contiguous()
        flat_d, dark_d = flat_d[:, lo:hi].contiguous(), dark_d[:, lo:hi].contiguous()
    r = tcp.Recon(ndet, w.nproj, nz, center, dtype, w.filter, 3)
    r.set_algorithm(alg)
    r.set_pad(pad)
    if tcfft:
        r.set_tcfft(tcfft)
    out = r.recon(raw_d, flat_d, dark_d, theta_d)
    torch.cuda.synchronize()
    out = out.float().cpu().numpy()
    r.close()
    sample = sorted({0, 1, nz // 2, nz - 1}) if nz > 4 else list(range(nz))
    raw_h = raw_d.view(torch.int16)[:, sample].contiguous().cpu().numpy().view(np.uint16)
    recon = orc.recon_padded if cut else orc.recon
    ref = recon(raw_h, flat_d[sample].cpu().numpy(), dark_d[sample].cpu().numpy(), w.theta, center, w.filter, 3, method, pad=pad)
    e2 = max(rl2(out[z], ref[i]) for i, z in enumerate(sample))
    em = max(float(np.abs(out[z] - ref[i]).max()) for i, z in enumerate(sample)) / float(np.abs(ref).max())
    gate = "1e-5 / -" if dtype == "f32" else "5e-3 / 1e-2"
    print("| %s | %d x %d^2, %d proj | %s | %d of %d | %.2e | %.2e | %s |" % (label, nz, ndet, w.nproj, dtype, len(sample), nz, e2, em, gate), flush=True)


def main():
    print("# Round 1: measured parity against the oracle (tests/parity_report.py)\n")
    print("Command (one B200): `python tests/parity_report.py`.  Gates: fp32 rel-L2 per slice <= 1e-5; fp16 rel-L2 <= 5e-3 and max-abs <= 1e-2 of")
    print("max |oracle| (north_star; asserted in tests/test_gpu_parity.py).\n")
    print("| case | chunk | dtype | slices compared | rel-L2 (max) | max-abs / max\\|oracle\\| | gate (rel-L2 / max-abs) |")
    print("|---|---|---|---|---|---|---|")
    w = sg.make_workload("C1")
    case("C1 FourierRec", w, list(range(8)), "f32")
    case("C1 FourierRec", w, list(range(8)), "f16")
    case("C1 FourierRec, edge padding", w, list(range(8)), "f32", pad="edge")
    case("C1 LineRec vs B_lin", w, list(range(8)), "f32", method="lin", alg="line")
    case("C1 LineRec vs B_lin", w, list(range(8)), "f16", method="lin", alg="line")
    w = sg.make_workload("C2")
    h = w.nz_total // 2
    case("C2 FourierRec", w, list(range(h - 4, h + 4)), "f32")
    case("C2 FourierRec", w, list(range(h - 4, h + 4)), "f16")
    case("C2, detector cut to 500 columns (tcp_create_det, padded to 512)", w, list(range(h - 4, h + 4)), "f32", cut=(6, 506))
    case("C2, detector cut to 333 columns (odd, object truncated)", w, list(range(h - 4, h + 4)), "f16", cut=(90, 423))
    w = sg.make_workload("C3")
    h = w.nz_total // 2
    case("C3 FourierRec (centre 515.5)", w, list(range(h - 8, h + 8)), "f16", gpu_inputs=True)
    w = sg.make_workload("C4")
    h = w.nz_total // 2
    case("C4 FourierRec (bench launch configuration)", w, list(range(h - 16, h + 16)), "f16", gpu_inputs=True)
    case("C4, row pass as DFT-as-GEMM on tcgen05 (opt-in)", w, list(range(h - 16, h + 16)), "f16", gpu_inputs=True, tcfft=4)
    w = sg.make_workload("C5")
    h = w.nz_total // 2
    case("C5 FourierRec (M = 8192, centre 2065.5, fp32 out)", w, list(range(h - 16, h + 16)), "f16_out32", gpu_inputs=True)


if __name__ == "__main__":
    main()
