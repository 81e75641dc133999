"""lasp_eval_grad_static: the allocation-free variant of lasp_eval_grad (scratch in a file-scope 16 MiB device array).

Collected last on purpose (the suite runs with `pytest -x`).  The GPU test passes alone in a fresh process and after the
other GPU tests: it builds its own contexts and depends on nothing they leave behind.
"""
import os
import re

import numpy as np
import pytest

from helpers import make, small_config, two_arm_config
from paper_2512_24840_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOL_GRAD, TOL_CONT, TOL_CHI2 = 1e-4, 1e-4, 1e-4          # the tolerances of tests/test_gpu_parity.py


def _body(src, name):
    """Source text of the extern "C" function `name` (up to the closing brace at column 0)."""
    a = src.index('extern "C" int ' + name + "(")
    return src[a:src.index("\n}\n", a)]


def test_static_entry_point_allocates_nothing():
    """The entry point's own body calls no allocating routine; the array is file-scope, aligned, of the size the header
    states; its address comes from cudaGetSymbolAddress (checked) at set-up, never from the host-side name."""
    src = open(os.path.join(ROOT, "paper_2512_24840_b200", "csrc", "lasp_gpu.cu")).read()
    hdr = open(os.path.join(ROOT, "include", "lasp_gpu.h")).read()
    body = _body(src, "lasp_eval_grad_static")
    assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|workspace\s*\(|\bnew\b|malloc\s*\(|std::vector", body)
    assert "lasp_static_scratch" not in body                     # host code uses the address kept in the ctx
    assert re.search(r"static __device__ __align__\(256\) float lasp_static_scratch\[LASP_STATIC_SCRATCH_BYTES", src)
    assert re.search(r"CUDA_TRY_C\(cudaGetSymbolAddress\(\(void \*\*\)&c->static_ws, lasp_static_scratch\)\)",
                     _body(src, "lasp_create"))
    assert re.search(r"#define LASP_STATIC_SCRATCH_BYTES \(16u << 20\)", hdr)


@pytest.mark.gpu
def test_static_entry_point_matches_eval_grad_twice(oracle_mod):
    """Two calls in a row on the shared array, the second on other spectra, a smaller batch and another model shape (so the
    array still holds the first call's planes): each equals lasp_eval_grad on the same inputs within the parity tolerances
    (the kernels are the same, so in fact bit for bit).  Then: linear-grid arms (per-pixel scratch), the streaming variant
    (global rows in the array), and a batch beyond the limit, which is refused with a clear error."""
    import torch
    from paper_2512_24840_b200 import binding, build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"

    def compare(m, case, params, n=None, **kw):
        sl = slice(0, n)
        args = (case["flux"][sl], case["ivar"][sl], case["mask"][sl], params[sl])
        ref = m.eval_grad(*args, **kw)
        got = m.eval_grad_static(*args, **kw)
        torch.cuda.synchronize()
        g, r = got["grad_u"].cpu().numpy().astype(np.float64), ref["grad_u"].cpu().numpy().astype(np.float64)
        assert np.isfinite(r).all()
        assert (np.abs(g - r).max(axis=1) / np.abs(r).max(axis=1)).max() <= TOL_GRAD
        assert np.allclose(got["chi2"].cpu().numpy(), ref["chi2"].cpu().numpy(), rtol=TOL_CHI2)
        assert np.allclose(got["cont"].cpu().numpy(), ref["cont"].cpu().numpy(), rtol=TOL_CONT, atol=1e-6)
        assert np.array_equal(got["status"].cpu().numpy(), ref["status"].cpu().numpy())
        assert np.array_equal(g, r)                                  # same kernels, same launch shape
        return got

    big = synth.make_case(1, oracle_mod.forward, B=70)              # 70: a ragged last group of four
    small = make(small_config(), oracle_mod, B=9)
    m1, m2 = binding.LaspModel(big["desc"]), binding.LaspModel(small["desc"])
    first = compare(m1, big, big["init"])                           # call 1
    compare(m2, small, small["init"])                               # call 2: other ctx, shorter rows, fewer spectra
    again = compare(m1, big, big["init"])                           # and the first once more: nothing leaked
    assert np.array_equal(first["grad_u"].cpu().numpy(), again["grad_u"].cpu().numpy())
    compare(m1, big, big["truth"], n=5)
    # against the oracle too (the existing path's own parity test, here through the new entry point)
    chi2, grad, _, st = oracle_mod.Oracle(big["desc"]).eval_grad(big["flux"], big["ivar"], big["mask"], big["init"])
    g = first["grad_u"].cpu().numpy().astype(np.float64)
    assert (np.abs(g - grad).max(axis=1) / np.abs(grad).max(axis=1)).max() <= TOL_GRAD
    assert np.allclose(first["chi2"].cpu().numpy(), chi2, rtol=TOL_CHI2) and np.array_equal(first["status"].cpu().numpy(), st)
    # caller-owned outputs: the wrapper allocates nothing either
    out = {k: torch.empty_like(v) for k, v in first.items()}
    m1.eval_grad_static(big["flux"], big["ivar"], big["mask"], big["init"], out=out)
    assert np.array_equal(out["grad_u"].cpu().numpy(), first["grad_u"].cpu().numpy())
    compare(m1, big, big["init"], variant=2)                        # streaming variant: T / a rows in the array
    arms = make(two_arm_config(), oracle_mod, B=11)                 # linear grid: per-pixel-kernel scratch planes
    m3 = binding.LaspModel(arms["desc"])
    compare(m3, arms, arms["init"])
    # beyond the limit: 16 MiB hold about 750 config-1 spectra
    n = 1200
    tile = lambda a: np.tile(a, (n // 70 + 1, 1))[:n]
    with pytest.raises(binding.LaspError, match="static array holds 16777216"):
        m1.eval_grad_static(tile(big["flux"]), tile(big["ivar"]), tile(big["mask"]), tile(big["init"]))
    compare(m1, big, big["init"])                                   # the refused call left the path usable
    for m in (m1, m2, m3):
        m.close()
