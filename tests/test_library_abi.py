"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, and exports every symbol
that include/lasp_gpu.h declares.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2512_24840_b200 import build
    return build.build()


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "lasp_gpu.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    txt = re.sub(r"#ifdef LASP_PHASE_TIMING.*?#endif", "", txt, flags=re.S)   # debug-build-only declarations
    return sorted(set(re.findall(r"\b(lasp_[a-z_]+)\s*\(", txt)))


def test_header_symbols_are_exported(libpath):
    L = ctypes.CDLL(libpath)
    syms = declared_symbols()
    assert "lasp_fit_batch" in syms and "lasp_eval_grad" in syms and len(syms) >= 9
    for s in syms:
        assert hasattr(L, s), s
    from paper_2512_24840_b200 import binding
    assert sorted(binding.SYMBOLS) == syms


def test_version_and_error_string(libpath):
    L = ctypes.CDLL(libpath)
    L.lasp_version.restype = ctypes.c_int
    assert L.lasp_version() >= 100
    L.lasp_last_error.restype = ctypes.c_char_p
    L.lasp_last_error.argtypes = [ctypes.c_void_p]
    assert isinstance(L.lasp_last_error(None), bytes)


def test_create_rejects_bad_arguments_without_gpu(libpath):
    from paper_2512_24840_b200 import binding
    L = binding.lib()
    out = ctypes.c_void_p()
    assert L.lasp_create(None, 0, ctypes.byref(out)) == -1  # LASP_ERR_INVALID_ARG
    d = binding.ModelDesc()
    assert L.lasp_create(ctypes.byref(d), 0, ctypes.byref(out)) == -1
    assert b"null" in L.lasp_last_error(None)


def test_binding_fails_loudly_without_cuda():
    import torch
    from paper_2512_24840_b200 import binding, synth
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    d = synth.make_model_desc(synth.CONFIGS[0]); d.pop("_rng")
    with pytest.raises(binding.LaspError):
        binding.LaspModel(d)


def test_sass_is_sm100(libpath):
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", libpath], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_library_reads_no_environment_variable():
    """Every switch is a field of lasp_fit_opts: nothing under csrc/ calls getenv."""
    csrc = os.path.join(ROOT, "paper_2512_24840_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_fit_opts_layout_matches_header():
    """The ctypes mirror of lasp_fit_opts has the header's fields in the header's order."""
    from paper_2512_24840_b200 import binding
    txt = open(os.path.join(ROOT, "include", "lasp_gpu.h")).read()
    body = re.search(r"typedef struct \{([^}]*)\} lasp_fit_opts;", txt, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            names += [n.strip() for n in decl.split(None, 1)[1].split(",")]
    assert names == [f[0] for f in binding.FitOpts._fields_]


def test_model_desc_layout_matches_header():
    """The ctypes mirror of lasp_model_desc has the header's fields in the header's order (pointers and scalars alike)."""
    from paper_2512_24840_b200 import binding
    txt = open(os.path.join(ROOT, "include", "lasp_gpu.h")).read()
    body = re.search(r"typedef struct \{([^}]*)\} lasp_model_desc;", txt, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            tail = decl.rsplit(None, 1)[0] if "," not in decl else decl
            parts = decl.replace("*", " ").split(",")
            names.append(parts[0].split()[-1])
            names += [p.strip() for p in parts[1:]]
    assert names == [f[0] for f in binding.ModelDesc._fields_]


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` times the oracle alone and prints one JSON line with the contract's keys."""
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0",
                          "--config", "0", "--ref-spectra", "8"], capture_output=True, text=True, cwd=ROOT, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert line["impl"] == "reference" and line["metric"] == "spectra fitted/sec (fixed Adam steps)" and line["value"] > 0
    assert line["gpu_launches"] == 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                          "--warmup", "0", "--config", "0", "--ref-spectra", "8"], capture_output=True, text=True, cwd=ROOT,
                         timeout=600, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""       # ranks other than 0 exit without work
