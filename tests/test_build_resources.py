"""The register / stack budget of the hot kernels, read from the built objects (cuobjdump --dump-resource-usage; no GPU).

The wide launch shape runs 768 threads per SM at 80 registers: the base variant of the transport kernel sits at the edge of
that budget, and a few more live values in its loop spill into local memory — measured on B200: an out-of-line call on the
(untaken) path of the NEXT-3 extensions took config 3s from 414 to 576 ms until it moved into the extras variant.  This test
holds the base variants to the stack they have today."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def resource_usage(obj):
    out = subprocess.run(["cuobjdump", "--dump-resource-usage", obj], capture_output=True, text=True, check=True).stdout
    res = {}
    for m in re.finditer(r"Function (\S+):\s*\n\s*REG:(\d+) STACK:(\d+)", out):
        res[m.group(1)] = (int(m.group(2)), int(m.group(3)))
    return res


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not on PATH")
def test_base_transport_kernels_keep_their_register_budget():
    from paper_2509_15377_b200 import build
    build.build()
    # <FK, HASB, TALLY, SMEMTAB, THREADS, TPB, BANDED, EXTRAS> of the five BASELINE configs' kernels
    cases = {"transport_fk1_b1.o": ("ILi1ELb1ELb1ELb1ELi768ELb0ELb0ELb0E", 80, 96),      # config 3: wide shape
             "transport_fk1_b0.o": ("ILi1ELb0ELb1ELb1ELi512ELb1ELb0ELb0E", 128, 48),     # configs 1, 2: latency shape
             "transport_fk2_b0.o": ("ILi2ELb0ELb1ELb1ELi512ELb1ELb0ELb0E", 128, 48),     # config 4
             "transport_fk0_b0.o": ("ILi0ELb0ELb1ELb1ELi512ELb1ELb0ELb0E", 128, 48)}     # config 5
    for obj, (pat, max_reg, max_stack) in cases.items():
        usage = resource_usage(os.path.join(build.OBJ_DIR, obj))
        hit = [(k, v) for k, v in usage.items() if "transport_kernel" in k and pat in k]
        assert len(hit) == 1, (obj, pat, list(usage)[:3])
        reg, stack = hit[0][1]
        assert reg <= max_reg and stack <= max_stack, (obj, reg, stack)
