"""Measured pipe numbers behind DESIGN.md 6.4: the tensor pipe (tcgen05.mma kind::tf32 with the narrow N the fit kernel's
table contractions would have) against the FP32 pipe (the kernel's own register block).  The probe is compiled here with
nvcc and run on the GPU box; the tcgen05 result is checked against numpy (small integers: exact in tf32)."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def probe(tmp_path_factory):
    import torch
    assert torch.cuda.is_available()
    so = str(tmp_path_factory.mktemp("probe") / "libpipe_probe.so")
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-shared", "-Xcompiler", "-fPIC",
                    "-o", so, os.path.join(HERE, "probes", "pipe_probe.cu")], check=True)
    L = ctypes.CDLL(so)
    L.probe_tcgen05.restype = ctypes.c_double
    L.probe_tcgen05.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_float)]
    L.probe_ffma.restype = ctypes.c_double
    L.probe_ffma.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int]
    L.probe_ffma2.restype = ctypes.c_double
    L.probe_ffma2.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int]
    return L


def expected(iters, n_tiles, n_cols):
    r, k, n = np.arange(128)[:, None], np.arange(8)[None, :], np.arange(n_cols)[:, None]
    B = (((2 * n + k) % 5) - 2).astype(np.float64)
    D = np.zeros((128, n_cols))
    for t in range(n_tiles):
        A = (((r + 3 * k + t) % 7) - 3).astype(np.float64)
        D += len(range(t, iters, n_tiles)) * (A @ B.T)
    return D


def test_tcgen05_tf32_narrow_n_against_ffma(probe, capsys):
    """tcgen05.mma M = 128, K = 8, kind::tf32, A and B from shared memory: cycles per MMA at N = 16 (8 spectra x [hi|lo])
    with the A tile fixed and with A streaming over 32 tiles, and at N = 256 for scale; the FP32 ceiling of the fit
    kernel's register block.  Numerics first: the accumulator must be the exact integer result."""
    rows = []
    for n_cols, n_tiles, n_acc in ((16, 1, 1), (16, 32, 1), (16, 32, 2), (16, 32, 4), (16, 32, 8), (16, 32, 16), (32, 32, 8),
                                   (64, 32, 8), (256, 1, 1), (256, 16, 2)):
        iters = 4096 + n_acc
        out = np.zeros(128 * n_cols, dtype=np.float32)
        cyc = probe.probe_tcgen05(iters, n_tiles, n_cols, n_acc, out.ctypes.data_as(ctypes.POINTER(ctypes.c_float)))
        assert cyc > 0, f"probe_tcgen05 failed with code {cyc}"
        assert np.array_equal(out.reshape(128, n_cols).astype(np.float64), expected(iters, n_tiles, n_cols)), (n_cols, n_tiles)
        mac = 128 * n_cols * 8 / cyc
        rows.append((n_cols, n_tiles, n_acc, cyc, mac))
    tf = probe.probe_ffma(296, 192, 20000)
    tf2 = probe.probe_ffma2(296, 192, 20000)
    assert tf > 30.0 and tf2 > 30.0
    lines = ["pipe probe (B200): tcgen05.mma.cta_group::1.kind::tf32, M=128, K=8, A/B from shared memory",
             "  N   A tiles  accumulators   cycles/MMA   MAC/clk/SM   useful MAC/clk/SM with [hi|lo] split operands (x 1/4)"]
    for n_cols, n_tiles, n_acc, cyc, mac in rows:
        lines.append(f"  {n_cols:3d}  {n_tiles:3d}      {n_acc:3d}         {cyc:8.2f}     {mac:8.1f}     {mac / 4:8.1f}")
    lines.append(f"FP32 pipe, acc[4][8] += p[g]*c[i] from registers, 296 x 192 threads: {tf:.1f} TFLOP/s "
                 f"= {tf * 1e12 / 2 / 148 / 1.965e9:.1f} FMA/clk/SM")
    lines.append(f"the same block with packed fma.rn.f32x2 (FFMA2, half the instructions): {tf2:.1f} TFLOP/s "
                 f"= {tf2 * 1e12 / 2 / 148 / 1.965e9:.1f} FMA/clk/SM")
    text = "\n".join(lines)
    with capsys.disabled():
        print("\n" + text)
    os.makedirs(os.path.join(os.path.dirname(HERE), "gpurun_out"), exist_ok=True)
    with open(os.path.join(os.path.dirname(HERE), "gpurun_out", "pipe_probe.txt"), "w") as f:
        f.write(text + "\n")
