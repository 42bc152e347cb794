"""include/lpc.h is a C header: a C99 client (tests/c_client/lpc_client.c) compiles against it with a C compiler and links
liblpc.so (no GPU needed for that); on the B200 the same program runs the five north-star calls from C and checks the
closed forms of PAPER.md Eq. 7 and Eq. 8 itself."""
import importlib.util
import os
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "c_client", "lpc_client.c")
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def _liblpc():
    spec = importlib.util.spec_from_file_location("_lpc_build", os.path.join(ROOT, "paper_2603_22553_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod.build()


def _compile(tmp_path):
    lib = _liblpc()
    exe = str(tmp_path / "lpc_client")
    libdir = os.path.dirname(lib)
    cmd = ["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-I" + os.path.join(ROOT, "include"),
           "-isystem", os.path.join(CUDA, "include"), SRC, "-o", exe, "-L" + libdir, "-llpc", "-L" + os.path.join(CUDA, "lib64"),
           "-lcudart", "-lm", "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(CUDA, "lib64")]
    subprocess.check_call(cmd)
    return exe


def test_header_compiles_as_c99_and_client_links(tmp_path):
    exe = _compile(tmp_path)
    assert os.path.exists(exe)
    # the header alone, strictest flags, as a translation unit of its own
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-fsyntax-only", "-x", "c",
                           os.path.join(ROOT, "include", "lpc.h")])


@pytest.mark.gpu
def test_c_client_runs_the_five_calls(tmp_path):
    exe = _compile(tmp_path)
    out = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    print(out.stdout, out.stderr)
    assert out.returncode == 0, out.stdout + out.stderr
    assert out.stdout.strip().endswith("OK")
