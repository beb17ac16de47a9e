"""Issue-port micro-benchmark (GPU): the evidence behind DESIGN.md section 7's statement that a packed f32x2 instruction holds the
issue port of an SM sub-partition for ~2 cycles and that nothing else issues in its shadow, so that the kernels' floor is
"issue cycles" = other instructions + ~2.2 x packed instructions (profiles/r2_issue_port_microbench.md holds a recorded run).
Compiles tests/microbench/issue_port.cu with nvcc for sm_100a and checks the two ratios the argument uses."""
import os
import re
import subprocess

import pytest

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def test_packed_f32x2_holds_the_issue_port_two_cycles(tmp_path):
    exe = str(tmp_path / "issue_port")
    subprocess.run(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-o", exe,
                    os.path.join(HERE, "microbench", "issue_port.cu")], check=True)
    out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout
    print(out)
    cyc = {}
    for line in out.splitlines():
        m = re.match(r"(.+?)\s+warps/SMSP (\d): .* -> ([\d.]+) cycles per warp-group", line)
        if m:
            cyc[(m.group(1).strip(), int(m.group(2)))] = float(m.group(3))
    for w in (4, 8):
        ffma2, ffma, iadd = cyc[("8 FFMA2", w)], cyc[("8 FFMA", w)], cyc[("8 IADD", w)]
        assert 1.8 * ffma <= ffma2 <= 2.6 * ffma                     # a packed instruction costs ~2 issue cycles
        both = cyc[("8 FFMA2 + 8 IADD", w)]
        assert both >= 0.9 * (ffma2 + iadd)                          # ... and ALU work does not issue in its shadow
        assert cyc[("8 MUFU + 56 IADD", w)] <= 1.15 * 64.0           # a MUFU costs one issue slot; its pipe is 1/8 rate
