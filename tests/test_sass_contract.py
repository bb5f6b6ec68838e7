"""The accumulation contract rounds every fp32 operation on its own.  ptxas 12.9
contracts `mul.rn.f32x2` + `add.rn.f32x2` into one FFMA2 even under --fmad=false and with the explicit .rn (found in
round 2 through a one-in-1e9 destination mismatch at n = 8), so the packed lerps of csrc/accumulate.cu form their
products with scalar FMULs.  This test reads the SASS of the built library and pins what must hold for that to stay
true: the pull kernel holds no FFMA2 besides the two of its division by a known reciprocal (fused by design), and the push
kernel holds exactly the four intended ones per instantiation (the folded index estimate, not a contract value).  CPU only (cuobjdump disassembles without a GPU)."""
import re
import shutil
import subprocess

import pytest

from paper_1809_03927_b200 import build


def _sass_by_function():
    lib = build.build()
    out = subprocess.run(["cuobjdump", "-sass", lib], check=True, capture_output=True, text=True).stdout
    funcs, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            funcs[name] = []
        elif name:
            funcs[name].append(line)
    return funcs


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not on PATH")
def test_no_unintended_packed_fma_in_the_contract_kernels():
    funcs = _sass_by_function()
    def count(kernel, op):
        names = [n for n in funcs if kernel in n]
        assert names, kernel
        return sum(len([l for l in funcs[n] if re.search(r"\b%s\b" % op, l)]) for n in names)
    # the pull kernel: only the two fmas of the known-reciprocal division (x, y packed), in its two kFastDiv instantiations
    assert count("dim_pull_kernel", "FFMA2") == 4
    # push_columns<checked, tile> x 4: Axy, A12z per cell and the x/y and z estimates per subvoxel
    assert count("emtm_push_kernel", "FFMA2") == 16 + 16 + 32  # runtime-nsz kernels (32 x 4 and 32 x 8 columns) + the nsz = 2 kernel (z-run unrolled twice)
    # the packed operations are really there (the kernels were built for sm_100a with f32x2)
    assert count("emtm_push_kernel", "FADD2") > 40 and count("dim_pull_kernel", "FADD2") > 4
    assert count("transport_kernel", "FFMA2") > 8
