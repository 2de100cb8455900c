"""Load-path probe (sldg_probe_load_rate, a diagnostic entry point): the rate at which the SMs pull the strided row
tiles the fused v passes gather, by TMA tensor copies, by 1-d TMA bulk copies and by plain 128-bit loads, with nothing
else going on.  DESIGN.md section 6 quotes these rates as the bound of the fused v passes; this test is the committed
micro-benchmark behind that statement (it prints a table, `pytest -s`, and writes gpurun_out/probe_load_rate.txt)."""
import os

import pytest
import torch

pytestmark = pytest.mark.gpu


def test_load_rate_of_strided_row_tiles():
    import paper_2110_14557_b200 as P
    if not torch.cuda.is_available():
        pytest.fail("gpu test without a CUDA device")
    g = P.Sldg(1, 1, [4, 4], 1, [0, 1.0, -1.0, 1.0])
    lines = []
    for label, X, R in (("HBM, 4.2 GB, row stride 512 kB (cfg4's X)", 64000, 8192), ("L2-resident, 33 MB", 4096, 1024)):
        src = torch.rand(R, X, dtype=torch.float64, device=g.device)
        for mode, name in ((0, "tensor copy"), (1, "bulk copy per row"), (2, "128-bit loads")):
            for wx, rows, depth, thr in ((16, 40, 8, 256), (16, 160, 8, 256), (16, 80, 4, 256), (32, 40, 4, 256), (8, 80, 8, 256), (64, 16, 8, 256)):
                if mode == 2 and rows * (wx // 2) > 4 * thr:
                    continue
                gbs = g.probe_load_rate(src, X, R, mode, wx, rows, depth if mode < 2 else 4, thr, max(1, (R // rows) // 4))
                lines.append(f"{label:44s} {name:18s} rows of {wx * 8:4d} B x {rows:3d}, depth {depth}: {gbs:8.1f} GB/s")
                assert gbs > 50.0
        del src
    out = "\n".join(lines)
    print("\n" + out)
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/probe_load_rate.txt", "w") as fh:
        fh.write(out + "\n")
