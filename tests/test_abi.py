"""C-ABI boundary checks that need no GPU: the library loads, exports every symbol that
include/rad.h declares, and rejects bad arguments before touching the device."""
import ctypes
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2501_03383_b200 import build, binding
    build.build()
    return binding.load()


def _declared_symbols():
    text = (ROOT / "include" / "rad.h").read_text()
    return sorted(set(re.findall(r"RAD_API[^;(]*?\b(rad_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_agree_on_symbols(lib):
    from paper_2501_03383_b200 import binding
    declared = _declared_symbols()
    assert len(declared) >= 10
    assert sorted(binding.ABI_SYMBOLS) == declared
    for name in declared:
        assert hasattr(lib, name), f"librad.so does not export {name}"


def test_only_abi_symbols_are_exported():
    import subprocess
    from paper_2501_03383_b200 import binding
    out = subprocess.run(["nm", "-D", "--defined-only", str(binding.LIB_PATH)],
                         capture_output=True, text=True, check=True).stdout
    exported = {ln.split()[-1] for ln in out.splitlines() if " T " in ln}
    assert {s for s in exported if s.startswith("rad_")} == set(binding.ABI_SYMBOLS)


def test_struct_layout_matches_header(tmp_path):
    """ctypes mirror of rad_config == what a C compiler makes of include/rad.h."""
    import subprocess
    from paper_2501_03383_b200 import binding
    src = tmp_path / "layout.c"
    src.write_text('''#include <stdio.h>
#include <stddef.h>
#include "rad.h"
int main(void){ printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n", sizeof(rad_config), offsetof(rad_config, n_dir),
  offsetof(rad_config, dirs), offsetof(rad_config, omega), offsetof(rad_config, dt),
  offsetof(rad_config, state_dtype), offsetof(rad_config, flags), offsetof(rad_config, window_origin),
  offsetof(rad_config, nyquist_factor), offsetof(rad_config, form_factor_type),
  offsetof(rad_config, form_factor_size)); return 0; }''')
    exe = tmp_path / "layout"
    subprocess.run(["gcc", "-I", str(ROOT / "include"), str(src), "-o", str(exe)], check=True)
    got = [int(x) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    c = binding.rad_config
    assert got == [ctypes.sizeof(c), c.n_dir.offset, c.dirs.offset, c.omega.offset, c.dt.offset,
                   c.state_dtype.offset, c.flags.offset, c.window_origin.offset, c.nyquist_factor.offset,
                   c.form_factor_type.offset, c.form_factor_size.offset]


def test_status_strings_and_version(lib):
    from paper_2501_03383_b200 import binding
    assert binding.status_string(0) == "RAD_OK"
    assert binding.status_string(binding.RAD_ERR_CUDA) == "RAD_ERR_CUDA"
    assert "sm_100a" in binding.rad_version()


GOOD_DIRS = np.array([[0.0, 0.0, 1.0], [1.0, 1.0, 0.0]])
GOOD_OMEGA = np.array([1e15, 2e15, 4e15])


@pytest.mark.parametrize("kw,msg", [
    (dict(dirs=np.array([[0.0, 0.0, 0.0]])), "direction"),
    (dict(dirs=np.array([[np.nan, 0.0, 1.0]])), "direction"),
    (dict(omega=np.array([2e15, 1e15])), "omega"),
    (dict(omega=np.array([0.0, 1e15])), "omega"),
    (dict(omega=np.array([1e15, np.inf])), "omega"),
    (dict(dt=0.0), "dt"),
    (dict(dt=float("nan")), "dt"),
    (dict(scale=-1.0), "scale"),
    (dict(state_dtype=7), "state_dtype"),
    (dict(flags=1 << 9), "flag"),
    (dict(form_factor=(7, (0, 0, 0))), "form_factor_type"),
    (dict(form_factor=("gaussian", (1e-8, float("inf"), 0))), "form_factor_size"),
    (dict(nyquist=-0.5), "nyquist_factor"),
    (dict(window=(5, (0, 0, 0), (1, 1, 1))), "window_type"),
])
def test_create_rejects_bad_arguments_without_a_device(lib, kw, msg):
    from paper_2501_03383_b200 import binding
    args = dict(dirs=GOOD_DIRS, omega=GOOD_OMEGA, dt=1e-17)
    args.update(kw)
    with pytest.raises(binding.RadError) as ei:
        binding.rad_create(**args)
    assert ei.value.status == binding.RAD_ERR_INVALID_ARG
    assert msg in str(ei.value)


def test_create_null_and_struct_size(lib):
    from paper_2501_03383_b200 import binding
    h = ctypes.c_void_p()
    assert lib.rad_create(None, ctypes.byref(h)) == binding.RAD_ERR_INVALID_ARG
    cfg = binding.rad_config(8, 0, 1, 1, 0, 0, 1e-17, 0.0, 0.0, 0, 0)
    assert lib.rad_create(ctypes.byref(cfg), ctypes.byref(h)) == binding.RAD_ERR_INVALID_ARG
    assert h.value is None
    lib.rad_destroy(None)  # NULL-safe
    assert lib.rad_launch_count(None) == 0


def test_no_cpu_fallback_without_gpu(lib):
    """On a box without a CUDA device a valid rad_create must fail loudly (RAD_ERR_CUDA)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2501_03383_b200 import binding
    with pytest.raises(binding.RadError) as ei:
        binding.rad_create(GOOD_DIRS, GOOD_OMEGA, 1e-17)
    assert ei.value.status == binding.RAD_ERR_CUDA


@pytest.mark.parametrize("kw,status,msg", [
    (dict(n_dir=257, n_omega=256), 5, "RAD_STATIC_MAX_BINS"),       # beyond the static scratch: RAD_ERR_UNSUPPORTED
    (dict(n_dir=0), 1, "n_dir"),
    (dict(out=0), 1, "out_device"),
    (dict(dt=0.0), 1, "dt"),
    (dict(scale=float("nan")), 1, "scale"),
    (dict(state_dtype=3), 1, "state_dtype"),
    (dict(n_particles=5, step_stride=4), 1, "step_stride"),
    (dict(n_particles=5, step_stride=5), 1, "NULL particle array"),
])
def test_spectrum_static_rejects_bad_arguments_without_a_device(lib, kw, status, msg):
    """rad_spectrum_static checks sizes and scalars before it touches the device (the pointers here are never read)."""
    from paper_2501_03383_b200 import binding
    a = dict(n_dir=2, n_omega=8, dt=1e-17, scale=1.0, state_dtype=binding.RAD_F32, n_particles=0, step_stride=0, out=256)
    a.update(kw)
    with pytest.raises(binding.RadError) as ei:
        binding.rad_spectrum_static(a["n_dir"], 256, a["n_omega"], 256, a["dt"], 0.0, a["scale"], a["state_dtype"], 0, 1,
                                    a["n_particles"], a["step_stride"], [0] * 10, a["out"])
    assert ei.value.status == status and msg in str(ei.value)


def test_spectrum_static_has_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    from paper_2501_03383_b200 import binding
    with pytest.raises(binding.RadError) as ei:
        binding.rad_spectrum_static(2, 256, 8, 256, 1e-17, 0.0, 1.0, binding.RAD_F32, 0, 1, 0, 0, [0] * 10, 256)
    assert ei.value.status == binding.RAD_ERR_CUDA


def test_product_path_never_touches_the_oracle():
    """The package must not import, read or link anything under oracle/ (or _work/)."""
    pkg = ROOT / "paper_2501_03383_b200"
    for p in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.h")):
        text = p.read_text()
        assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), p
        assert "rad_oracle" not in text and "_work/" not in text, p


def _build_c_client(tmp_path):
    import subprocess
    from paper_2501_03383_b200 import binding, build
    build.build()
    exe = tmp_path / "rad_client"
    subprocess.run(["gcc", "-std=c11", "-Wall", "-Werror", "-I", str(ROOT / "include"), str(ROOT / "tests" / "rad_client.c"),
                    "-L", str(binding.LIB_PATH.parent), "-lrad", "-lm", "-o", str(exe)], check=True)
    import os
    env = dict(os.environ, LD_LIBRARY_PATH=str(binding.LIB_PATH.parent) + ":" + os.environ.get("LD_LIBRARY_PATH", ""))
    return subprocess.run([str(exe)], capture_output=True, text=True, env=env)


def test_c_client_compiles_against_the_header_and_fails_loudly_without_a_gpu(tmp_path):
    """tests/rad_client.c: include/rad.h is a plain C11 header (-Wall -Werror), the program links against
    librad.so alone (no torch, no Python, no CUDA headers), and without a CUDA device rad_create reports
    RAD_ERR_CUDA -- no CPU fallback.  (On a GPU box the same binary runs the path: see the gpu test.)"""
    res = _build_c_client(tmp_path)
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        assert res.returncode == 0 and "rad_client OK" in res.stdout, res.stdout + res.stderr
    else:
        assert res.returncode == 2 and "RAD_ERR_CUDA" in res.stderr, res.stdout + res.stderr


@pytest.mark.gpu
def test_c_client_runs_the_abi_from_plain_c(tmp_path):
    """The whole path (host buffers in, spectrum out) driven from plain C against a closed form."""
    res = _build_c_client(tmp_path)
    assert res.returncode == 0 and "rad_client OK" in res.stdout, res.stdout + res.stderr
    print(res.stdout.strip())
