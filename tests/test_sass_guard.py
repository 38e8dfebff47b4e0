"""A guard on the built library's SASS (host tool only, no GPU): every packed FMA of the push kernels that
carry the headline -- sub-blocks of 24 samples, the two section forms of a Butterworth band-pass, with and
without the trigger, both layouts, aligned and shifted rows -- takes its table operand from a UNIFORM
register, and none of them spills.  DESIGN.md 6/7: an FFMA2 with three register-file operands runs at two
thirds of the rate, and ptxas gives up the uniform path for a whole kernel at small provocations (a
section index needed in a vector register, an atomic intrinsic, register pressure): measured -30 %, silently.
Skipped where cuobjdump is not installed."""
import collections
import re
import shutil
import subprocess

import pytest

from paper_2605_20132_b200 import build as fbuild


@pytest.fixture(scope="module")
def kernels():
    tool = shutil.which("cuobjdump") or shutil.which("/usr/local/cuda/bin/cuobjdump")
    if tool is None:
        pytest.skip("cuobjdump not installed")
    fbuild.build_library()
    from paper_2605_20132_b200 import stream
    txt = subprocess.run([tool, "-sass", stream.library_path()], capture_output=True, text=True, check=True).stdout
    out = {}
    for f in re.split(r"\n\s*Function : ", txt)[1:]:
        name = f.split("\n")[0]
        # filark_push_cm_kernel<L, CTAS, kForm, kTM, kDyn, kShift>
        m = re.search(r"filark_push_cm_kernelILi(\d+)ELi(\d)ELi(\d)ELb(\d)ELb(\d)ELb(\d)", name)
        mt = re.search(r"filark_push_tr_kernelILi(\d)", name)       # time-major, one channel per lane: <kForm>
        if not m and not mt:
            continue
        ffma2 = [ln for ln in f.split("\n") if "FFMA2" in ln]
        ops = collections.Counter(mm.group(1).split(".")[0] for mm in re.finditer(r"\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", f))
        key = tuple(int(g) for g in m.groups()) if m else ("tr", int(mt.group(1)))
        out[key] = dict(ffma2=len(ffma2), uniform=sum("UR" in ln for ln in ffma2),
                                                      spills=ops["STL"] + ops["LDL"])
    return out


def test_headline_kernels_keep_uniform_operands_and_do_not_spill(kernels):
    assert len(kernels) >= 40                        # every instantiation was found
    lean = {k: v for k, v in kernels.items() if k[0] == 24 and k[2] in (0, 2)}
    assert len(lean) >= 16
    for key, v in lean.items():
        assert v["ffma2"] >= 300, key                # 8 sections x 24 samples x (local pass + fix-up), STA/LTA
        assert v["uniform"] == v["ffma2"], f"{key}: {v['ffma2'] - v['uniform']} FFMA2 with a register-file table operand"
        assert v["spills"] == 0, f"{key}: local-memory spills"


def test_every_form_at_24_samples_is_uniform_too(kernels):
    assert ("tr", 0) in kernels and ("tr", 1) in kernels
    for key, v in kernels.items():
        if key[0] in (24, "tr"):
            assert v["uniform"] == v["ffma2"] and v["spills"] == 0, key
