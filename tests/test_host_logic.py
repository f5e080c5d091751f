"""CPU-only checks of the product's host side: the library builds, loads and exports the whole C ABI;
the fast-division helper used for site index -> coordinates is exact (brute force, host compile)."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    import paper_1801_01473_b200 as lq
    from paper_1801_01473_b200.build import build
    build()
    header = open(os.path.join(ROOT, "include", "lqcd.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(lqcd_[a-z_0-9]+)\s*\(", header))
    declared.discard("lqcd_ctx")
    assert len(declared) >= 19
    assert declared == set(lq.EXPORTS), declared ^ set(lq.EXPORTS)
    lib = lq.load_library()                      # dlopen works without a GPU (libcudart only)
    for name in declared:
        assert getattr(lib, name) is not None


def test_create_fails_loudly_without_a_gpu_or_on_bad_extents():
    import torch
    import paper_1801_01473_b200 as lq
    assert not lq.lqcd_create(3, 4, 4, 4)
    assert "even" in lq.lqcd_last_error(None)
    if not torch.cuda.is_available():
        assert not lq.lqcd_create(4, 4, 4, 4)    # no device: NULL, never a CPU fallback
        assert "CUDA" in lq.lqcd_last_error(None)
        with pytest.raises(RuntimeError):
            lq.Lattice((4, 4, 4, 4))


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1801_01473_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in text.lower().replace("no cpu fallback", ""), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "import paper_1801_01473_b200" not in text and "liblqcd_b200" not in text


def test_fastdiv_is_exact(tmp_path):
    src = tmp_path / "fd.cpp"
    src.write_text(r'''
#include "fastdiv.h"
#include <cstdio>
#include <cstdint>
int main() {
    uint64_t s = 88172645463325252ull;
    for (uint32_t d = 1; d <= 4100; ++d) {
        FastDiv f = make_fastdiv(d);
        for (uint32_t n = 0; n < 70000; ++n) if (fastdiv(n, f) != n / d) { printf("bad %u %u\n", n, d); return 1; }
        for (int i = 0; i < 2000; ++i) {
            s ^= s << 13; s ^= s >> 7; s ^= s << 17;
            uint32_t n = (uint32_t)(s >> 33);             // < 2^31
            if (fastdiv(n, f) != n / d) { printf("bad %u %u\n", n, d); return 1; }
        }
        uint32_t edge[] = {0x7fffffffu, 0x7ffffffeu, (0x7fffffffu / d) * d, (0x7fffffffu / d) * d - 1};
        for (uint32_t n : edge) if (n < 0x80000000u && fastdiv(n, f) != n / d) { printf("bad %u %u\n", n, d); return 1; }
    }
    puts("ok");
    return 0;
}
''')
    exe = tmp_path / "fd"
    inc = os.path.join(ROOT, "paper_1801_01473_b200", "csrc")
    subprocess.run(["g++", "-O2", "-I", inc, "-o", str(exe), str(src)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True)
    assert out.stdout.strip() == "ok"


def test_ncu_traffic_constants_of_bench_match_the_profile_they_cite():
    """bench.py reports `roofline.traffic` from a constant measured once under `ncu --set full`; the constant and
    the file it names must say the same thing (it would otherwise go stale silently when the kernel changes)."""
    sys.path.insert(0, ROOT)
    import bench
    unit = {"Gbyte": 1.0, "Mbyte": 1e-3, "Kbyte": 1e-6, "byte": 1e-9}
    assert bench.NCU_DRAM_GB_PER_LAUNCH
    for (workload, recon), (rd, wr, path) in bench.NCU_DRAM_GB_PER_LAUNCH.items():
        text = open(os.path.join(ROOT, path)).read()
        m = re.search(r"dslash_kernel<double, %d(?:, 0)+>.*?dram__bytes_read\.sum\s+([0-9.]+) (\w+).*?"
                      r"dram__bytes_write\.sum\s+([0-9.]+) (\w+)" % recon, text, flags=re.S)
        assert m, (workload, recon, path)
        assert abs(float(m.group(1)) * unit[m.group(2)] - rd) <= 1e-5 * rd
        assert abs(float(m.group(3)) * unit[m.group(4)] - wr) <= 1e-5 * wr
