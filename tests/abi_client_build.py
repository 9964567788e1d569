"""Compile tests/abi_client.c (a plain C99 user of include/rfoe.h) with gcc against librfoe.so and the CUDA runtime."""
import os
import subprocess

import paper_2301_04642_b200 as rfoe

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def build(outdir) -> str:
    rfoe.load_library()                                   # builds librfoe.so first if the sources are newer
    pkg = os.path.join(ROOT, "paper_2301_04642_b200")
    exe = os.path.join(str(outdir), "abi_client")
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-Wextra", "-pedantic", "-Werror",
           "-I", os.path.join(ROOT, "include"), "-isystem", os.path.join(CUDA, "include"),
           os.path.join(ROOT, "tests", "abi_client.c"), "-o", exe,
           "-L", pkg, "-l:librfoe.so", "-L", os.path.join(CUDA, "lib64"), "-lcudart", "-lm",
           f"-Wl,-rpath,{pkg}", f"-Wl,-rpath,{os.path.join(CUDA, 'lib64')}"]
    subprocess.run(cmd, check=True, cwd=ROOT)
    return exe
