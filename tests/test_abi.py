"""CPU-side checks of the boundary: the CUDA library builds for sm_100a, loads without a GPU, and
exports every symbol include/qmc_b200.h declares (no compute calls here)."""
import ctypes
import os
import re
import subprocess

import pytest

from paper_1802_06922_b200 import api, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "qmc_b200.h")


def declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qmc_[a-z_0-9]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    build.build_library()
    return api.load_library()


def test_header_declares_the_six_calls():
    names = declared_functions()
    for n in ["qmc_spline_create", "qmc_spo_vgl", "qmc_det_init", "qmc_det_ratio", "qmc_det_accept_update",
              "qmc_sweep"]:
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    names = declared_functions()
    assert sorted(api.EXPORTS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "qmc_b200.h"\nint main(void){qmc_sweep_opts_t o = {0}; return o.iel_begin + QMC_OK;}\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_sweep_opts_layout_matches_binding():
    # the ctypes mirror must have the C struct's size and offsets: compile the header and ask the compiler
    src = "#include <stdio.h>\n#include <stddef.h>\n#include \"qmc_b200.h\"\nint main(void){printf(\"%zu %zu %zu %zu %zu %zu\\n\", sizeof(qmc_sweep_opts_t), offsetof(qmc_sweep_opts_t, phi_record), offsetof(qmc_sweep_opts_t, force_out), offsetof(qmc_sweep_opts_t, drift_tau), offsetof(qmc_sweep_opts_t, rprop_out), offsetof(qmc_sweep_opts_t, fcur_out));return 0;}\n"
    import tempfile
    with tempfile.TemporaryDirectory() as tmp:
        c = os.path.join(tmp, "t.c")
        with open(c, "w") as f:
            f.write(src)
        exe = os.path.join(tmp, "t")
        subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        got = [int(v) for v in subprocess.run([exe], capture_output=True, text=True, check=True).stdout.split()]
    S = api.SweepOpts
    assert got == [ctypes.sizeof(S), S.phi_record.offset, S.force_out.offset, S.drift_tau.offset, S.rprop_out.offset,
                   S.fcur_out.offset]


def test_built_for_sm_100a():
    out = subprocess.run(["cuobjdump", "-lelf", api.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_error_paths_without_gpu(lib):
    # NULL handles are rejected before any CUDA call
    assert lib.qmc_spline_info(None, None, None) == -1
    assert b"NULL" in lib.qmc_last_error()
    assert lib.qmc_det_flush(None, None) == -1
    assert lib.qmc_launch_count() >= 0
