"""Helper of the ABI tests: compiles tests/abi_consumer.c (plain C99) against libzfac.so and the CUDA runtime."""
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def compile_consumer(out: str) -> str:
    lib_dir = os.path.join(ROOT, "paper_2404_19163_b200")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    cmd = ["gcc", "-std=c99", "-Wall", "-Werror", f"-I{os.path.join(ROOT, 'include')}", f"-I{cuda}/include",
           os.path.join(ROOT, "tests", "abi_consumer.c"), "-o", out, f"-L{lib_dir}", "-lzfac", f"-L{cuda}/lib64", "-lcudart",
           "-lm", f"-Wl,-rpath,{lib_dir}", f"-Wl,-rpath,{cuda}/lib64"]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    return out
