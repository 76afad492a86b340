"""The grid barrier of the persistent step kernel has no L1 invalidation on its waiting side (
`grid_barrier` in csrc/ts_api.cu).  That is sound only while NO instantiation of that kernel reads, through L1,
anything a thread may write during a launch.  This test holds the kernel to it by reading the machine code of the
built library: every global load of every `k_persistent` instantiation must be either a gpu-scope strong load
(`LDG.E...STRONG.GPU`: `ld.global.cg` / `ld.relaxed.gpu`, served at L2) or a non-coherent load of launch-constant data
(`LDG.E...CONSTANT`: `ld.global.nc` / `__ldg`), and the barrier must be there as `MEMBAR.ALL.GPU` + `REDG` with no
`CCTL.IVALL`.  A plain `LDG.E` (an L1-cached weak load) that slips into a new code path fails here, on the CPU."""
import re
import shutil
import subprocess

import pytest

from paper_1807_01148_b200 import build


def _sass():
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    try:
        out = subprocess.run([cuobjdump, "-sass", build.build()], capture_output=True, text=True, check=True).stdout
    except (OSError, subprocess.CalledProcessError) as e:      # no toolkit on this machine
        pytest.skip(f"cuobjdump unavailable: {e}")
    functions, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            functions[name] = []
        elif name and "/*" in line:
            functions[name].append(line)
    return functions


def test_persistent_kernel_reads_mutable_data_at_l2_only():
    functions = {n: body for n, body in _sass().items() if "k_persistent" in n}
    assert len(functions) >= 20, "5 CTA sizes x EMIS x EXT instantiations expected"
    for name, body in functions.items():
        loads = [l for l in body if re.search(r"\bLDG\.", l) or re.search(r"\bLD\.E", l)]
        assert loads, name
        for l in loads:
            op = re.search(r"\b(LDG?\.[A-Z0-9_.]+)", l).group(1)
            assert "STRONG.GPU" in op or "CONSTANT" in op, f"{name}: L1-cached weak load {op} -- see grid_barrier"
        text = "\n".join(body)
        assert "CCTL.IVALL" not in text and "MEMBAR.SC" not in text, f"{name}: a __threadfence() is back in the step loop"
        assert "MEMBAR.ALL.GPU" in text and "REDG.E.ADD.STRONG.GPU" in text, f"{name}: the barrier's release is gone"
