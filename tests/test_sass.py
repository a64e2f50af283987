"""Static checks of the built library's machine code (cuobjdump -sass; no GPU needed).

1. The kernels of one generation run under programmatic dependent launch (csrc/pdl.cuh): a kernel may start while its
   predecessor is still writing.  ld.global.nc (SASS LDG.*.CONSTANT, what __ldg and `const __restrict__` compile to) is
   only legal for data that is read-only for the kernel's whole lifetime, so buffers written by an earlier kernel of the
   chain (population, fitness, partial sums, W images and scales, rank / prefix tables, stop flag) must be read with
   coherent loads.  Only the knowledge base X, t (never written by a kernel) may use the non-coherent path.
2. The tensor-core kernel really is one: tcgen05.mma (UTCHMMA), TMEM loads (LDTM) and the bulk-copy engine (UBLKCP)."""
import os
import re
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1211_5481_b200", "csrc")


@pytest.fixture(scope="module")
def sass():
    from paper_1211_5481_b200 import build
    lib = build.build()
    exe = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(exe):
        pytest.skip("cuobjdump not available")
    txt = subprocess.run([exe, "-sass", lib], capture_output=True, text=True, check=True).stdout
    funcs = {}
    for part in re.split(r"Function : ", txt)[1:]:
        name, _, body = part.partition("\n")
        funcs[name.strip()] = body
    return funcs


def _find(funcs, needle):
    hits = [(k, v) for k, v in funcs.items() if needle in k]
    assert hits, f"no kernel named *{needle}* in libgame.so"
    return hits


CHAIN_KERNELS_WITHOUT_KB = ["build_w_images_kernel", "row_scale_kernel", "finalize_fitness_kernel", "ga_step_kernel",
                            "rank_kernel", "roulette_prefix_kernel"]


@pytest.mark.parametrize("kernel", CHAIN_KERNELS_WITHOUT_KB)
def test_chain_kernels_use_no_noncoherent_loads(sass, kernel):
    for name, body in _find(sass, kernel):
        bad = re.findall(r"LDG\.[A-Z0-9.]*CONSTANT[^\n]*", body)
        assert not bad, f"{name}: non-coherent loads of buffers written inside the launch chain: {bad[:3]}"
        assert re.search(r"\bLDG\.", body), f"{name}: expected global loads"


def test_fitness_kernels_keep_noncoherent_loads_for_the_knowledge_base_only(sass):
    """The fused fitness kernels read X and t through the non-coherent path and W / scales / partial sums / stop flag
    coherently: at least four coherent loads each, and in the source every __ldg names X or t."""
    for name, body in _find(sass, "fitness_umma_kernel") + _find(sass, "fitness_ffma_kernel"):
        coherent = [l for l in re.findall(r"\bLDG\.[^\n]*", body) if "CONSTANT" not in l]
        assert len(coherent) >= 2, name
    for fn in ("fitness_umma.cuh", "fitness_ffma.cuh", "ga_kernels.cuh"):
        for i, line in enumerate(open(os.path.join(CSRC, fn)), 1):
            code = line.split("//")[0]
            if "__ldg(" in code:
                assert re.search(r"__ldg\((prm\.t|t \+|row|xr|reinterpret_cast<const float4\*>\(row\))", code), f"{fn}:{i}: {line.strip()}"
    # the kernels of the chain take their chain-written inputs as plain pointers
    src = open(os.path.join(CSRC, "ga_kernels.cuh")).read()
    sig = src[src.index("ga_step_kernel(const float* W"):][:200]
    assert "__restrict__" not in sig


def test_tensor_kernel_is_tcgen05(sass):
    hits = _find(sass, "fitness_umma_kernel")
    assert len(hits) == 6                                   # 2 expansions x 3 activations
    for name, body in hits:
        assert body.count("UTCHMMA") >= 3, name             # three MMAs per K step (F16X3)
        assert "LDTM" in body and "UBLKCP" in body and "UTCBAR" in body, name
