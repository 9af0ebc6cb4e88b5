"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/radiusfps.h declares; the Python binding marshals and validates without a GPU."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_06255_b200 import build
    return ctypes.CDLL(build.build())


def declared_functions():
    text = open(os.path.join(ROOT, "include", "radiusfps.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fps_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("fps_index_build", "fps_sample", "fps_index_destroy", "fps_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in declared_functions():
        assert hasattr(lib, name), name


def test_binding_lists_every_declared_symbol():
    from paper_2606_06255_b200 import binding
    assert sorted(binding.EXPORTS) == declared_functions()


def test_struct_layouts_match_header(tmp_path):
    """Every field of fps_build_opts / fps_stats sits at the same offset in the ctypes binding as in the C header:
    a small C program compiled against include/radiusfps.h prints sizeof and offsetof of every field."""
    import subprocess
    from paper_2606_06255_b200 import binding
    prog = ["#include <stdio.h>", "#include <stddef.h>", '#include "radiusfps.h"', "int main(void) {"]
    for cname, cls in (("fps_build_opts", binding.fps_build_opts), ("fps_stats", binding.fps_stats)):
        prog.append(f'printf("{cname} %zu\\n", sizeof({cname}));')
        for field, _ in cls._fields_:
            prog.append(f'printf("{cname}.{field} %zu\\n", offsetof({cname}, {field}));')
    prog += ["return 0; }"]
    src, exe = tmp_path / "layout.c", tmp_path / "layout"
    src.write_text("\n".join(prog))
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    want = dict(line.split() for line in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines())
    for cname, cls in (("fps_build_opts", binding.fps_build_opts), ("fps_stats", binding.fps_stats)):
        assert ctypes.sizeof(cls) == int(want[cname]), cname
        for field, _ in cls._fields_:
            assert getattr(cls, field).offset == int(want[f"{cname}.{field}"]), (cname, field)
    # and the header has no field the binding lacks
    text = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "radiusfps.h")).read(), flags=re.S)
    body = text[text.index("typedef struct {", text.index("fps_build_opts;")):text.index("} fps_stats;")]
    names = [n.strip() for decl in re.findall(r"int(?:32|64)_t\s+([^;]+);", body) for n in decl.split(",")]
    assert names == [f for f, _ in binding.fps_stats._fields_]


def test_version_and_error_strings(lib):
    lib.fps_version.restype = ctypes.c_char_p
    lib.fps_last_error.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.fps_version()
    assert lib.fps_last_error() == b""


def test_null_and_bad_arguments_fail_without_a_gpu(lib):
    lib.fps_index_build.restype = ctypes.c_void_p
    lib.fps_last_error.restype = ctypes.c_char_p
    assert lib.fps_index_build(None, 10, 1) is None
    assert b"NULL" in lib.fps_last_error()
    assert lib.fps_last_status() == -1
    buf = (ctypes.c_float * 3)()
    assert lib.fps_index_build(buf, 0, 1) is None
    assert lib.fps_sample(None, 1, 0, None, None, None) == -1
    assert lib.fps_sample_host(buf, 1, 1, 2, 0, buf, buf, None) == -1      # M > N
    lib.fps_index_destroy(None)                                             # allowed


def test_binding_rejects_host_tensor_and_wrong_dtype():
    from paper_2606_06255_b200 import binding
    with pytest.raises(ValueError):
        binding.fps_index_build(torch.zeros(8, 3))                 # not on a CUDA device
    with pytest.raises(ValueError):
        binding._check_points(torch.zeros(8, 3, dtype=torch.float64))
    with pytest.raises(ValueError):
        binding._check_points(torch.zeros(8, 4))
    assert binding._check_points(torch.zeros(2, 8, 3)) == (2, 8)


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_06255_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "oracle/" not in src or f == "inputs.py" or "Nothing here is used by" in src, f


def test_no_packed_fma_in_the_built_kernels():
    """The one distance expression must never be contracted to FMA (BASELINE.json north_star).  The
    scalar path uses __f*_rn intrinsics; the packed path (FADD2/FMUL2 in the candidate-set FPS) must
    not contain FFMA2, which ptxas would produce from mul.f32x2 + add.f32x2 even under --fmad=false."""
    import shutil
    import subprocess
    from paper_2606_06255_b200 import build
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", build.build()], capture_output=True, text=True, check=True).stdout
    assert "FMUL2" in sass                      # the packed path is really there
    assert "FFMA2" not in sass
    # scalar FFMA may only come from the sqrt_rn / division sequences (MUFU + Newton steps and their fix-up
    # subroutines), never from a distance: per kernel at most a handful per MUFU, and always fewer than the
    # FMUL of the distances
    fn, counts = None, {}
    for line in sass.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            fn = m.group(1)
            counts[fn] = [0, 0, 0]
        elif fn and " FFMA" in line:
            counts[fn][0] += 1
        elif fn and (" FMUL " in line or " FMUL2 " in line):
            counts[fn][1] += 1
        elif fn and " MUFU." in line:
            counts[fn][2] += 1
    checked = 0
    for fn, (ffma, fmul, mufu) in counts.items():
        # the Euclidean-mode instantiations (fourth template flag = true) evaluate sqrt_rn at every update:
        # their FFMA are the Newton steps of those square roots; the squared-mode kernels have none there
        # (k_fps_whole: third template argument)
        euclid = re.search(r"k_fps_batchedILi\d+ELi\d+ELb[01]ELb1ELb[01]EE|k_fps_wholeILi\d+ELb[01]ELb1EE", fn) is not None
        if "k_fps_" in fn and not euclid:
            assert ffma <= 8 * mufu + 16 and fmul > ffma, (fn, ffma, fmul, mufu)
            checked += 1
    assert checked >= 10


def test_every_build_kernel_waits_for_its_predecessor_grid():
    """The index build chains its kernels by programmatic dependent launch: the order of
    memory operations is the stream order only if EVERY kernel launched that way starts with grid_dep_sync()
    (griddepcontrol.wait before its first memory access), and no build kernel is launched around launch_pdl."""
    src = open(os.path.join(ROOT, "paper_2606_06255_b200", "csrc", "index_build.cu")).read()
    kernels = re.findall(r"__global__\s+void\s+(?:__launch_bounds__\([^)]*\)\s*)?(k_\w+)\s*\(", src)
    assert len(kernels) >= 16
    for k in kernels:
        body = src[re.search(r"__global__\s+void\s+(?:__launch_bounds__\([^)]*\)\s*)?" + k + r"\s*\(", src).end():]
        first = body[body.index("{") + 1:].lstrip().splitlines()[0].strip()
        assert first == "grid_dep_sync();", (k, first)
    assert "<<<" not in src.replace("// ", ""), "a build kernel is launched without launch_pdl"
    assert set(re.findall(r"launch_pdl(?:_smem|_cluster)?\(log, (?:[^,(]+\([^)]*\), )?(?:\w+, )?(k_\w+),", src)) == set(kernels)
    helper = src[src.index("void grid_dep_sync()"):]
    helper = helper[:helper.index("}")]
    assert helper.index("griddepcontrol.launch_dependents") < helper.index("griddepcontrol.wait")
