"""Static checks on the SASS of libsw.so (no GPU needed; skipped when cuobjdump is not installed).

Programmatic dependent launch: a kernel launched as a programmatic dependent may run while its predecessor still
does, and may read what earlier kernels of the stream wrote only after griddepcontrol.wait (SASS: ACQBULK).  ptxas
does not order ld.global.nc loads (__ldg, const __restrict__ parameters) against that instruction: it once moved the
loads of count[seq] / seqlens[seq] of the decode attention kernel above it, and the kernel read block lists the
selection had not finished writing (a wrong output or a wild address, about one run in four of the cfg 3 test).  The
failure depends on timing, so the property is checked where it is decided: in the instruction order."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LIB = os.path.join(ROOT, "paper_2602_07397_b200", "libsw.so")
CUOBJDUMP = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"

# kernels of the decode chain that read their predecessors' output; nothing may be loaded from global memory before
# the wait.  (decode_tail_kernel is not listed: its prologue reads seqlens and tau, which are written before the
# selection's first kernel passes its own wait -- see decode_tail.cu.)
PDL_KERNELS = ["attn_decode_kernel", "attn_decode_merge_kernel", "decode_stream_kernel", "decode_duty_kernel"]


def sass_functions():
    out = subprocess.run([CUOBJDUMP, "-sass", LIB], capture_output=True, text=True, check=True).stdout
    funcs, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
        elif name is not None:
            m = re.match(r"\s+/\*[0-9a-f]+\*/\s+(.*?);", line)
            if m:
                funcs[name].append(m.group(1).strip())
    return funcs


@pytest.mark.skipif(not os.path.exists(CUOBJDUMP), reason="cuobjdump not installed")
def test_no_global_load_is_scheduled_above_griddepcontrol_wait():
    if not os.path.exists(LIB):
        pytest.skip("libsw.so not built")
    funcs = sass_functions()
    checked = 0
    for fname, insts in funcs.items():
        if not any(k in fname for k in PDL_KERNELS):
            continue
        waits = [i for i, s in enumerate(insts) if "ACQBULK" in s]
        assert waits, f"{fname}: no griddepcontrol.wait (ACQBULK) in a kernel of the programmatic-dependent chain"
        early = [s for s in insts[:waits[0]] if re.search(r"\b(LDG|LDGSTS|LD\.E|ATOMG|RED)\b", s.split()[0] if not s.startswith("@") else s.split()[1])]
        assert not early, f"{fname}: global loads above griddepcontrol.wait: {early[:4]}"
        checked += 1
    assert checked >= len(PDL_KERNELS)
