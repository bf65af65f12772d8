"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/mlp_pipe.h declares; the ctypes structs match the header; argument errors are reported
without a GPU.  No compute call is made here."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "mlp_pipe.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mlp_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    fns = _declared_functions()
    for need in ["mlp_pipe_create", "mlp_pipe_run", "mlp_pipe_destroy", "mlp_pipe_create_chain", "mlp_pipe_run_chain",
                 "mlp_pipe_run_host", "mlp_pipe_stats", "mlp_pipe_hidden"]:
        assert need in fns


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2607_07862_b200 import binding, build

    path = build.build_lib()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for fn in _declared_functions():
        assert hasattr(lib, fn), f"{fn} declared in mlp_pipe.h but not exported"
    assert sorted(binding.EXPORTS) == _declared_functions()
    assert b"sm_100a" in binding.load().mlp_pipe_version()


def test_sass_is_blackwell_native():
    """tcgen05.mma -> UTCHMMA, tcgen05.ld -> LDTM, TMA -> UTMALDG, protocol -> REDG/LDG .STRONG.GPU."""
    from paper_2607_07862_b200 import build

    cuobjdump = "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not installed")
    sass = subprocess.run([cuobjdump, "-sass", build.build_lib()], capture_output=True, text=True).stdout
    for mnemonic in ["UTCHMMA", "LDTM", "UTMALDG", "REDG.E.ADD.STRONG.GPU", "LDG.E.STRONG.GPU"]:
        assert mnemonic in sass, mnemonic
    assert "HMMA." not in sass.replace("UTCHMMA", ""), "legacy mma.sync path must not be present"
    # the GeLU epilogue runs on the packed fp32 pipe: 5 packed operations per 2 tanh (cfg 2 anatomy)
    packed, tanh = len(re.findall(r"\b(?:FMUL2|FFMA2)\b", sass)), sass.count("MUFU.TANH")
    assert tanh > 0 and packed * 2 == tanh * 5, (packed, tanh)


def test_mma_issue_loop_has_no_per_instruction_elect_loops():
    """The MMA warp runs converged and issues under elect.sync ("The MMA issuer paces the tensor pipe"): every
    UTCHMMA of the kernel must be straight-line code.  A `lane == 0` thread would make ptxas wrap each one into an ELECT / BRA.U.ANY
    loop over the active lanes, which is what paced the tensor pipe before."""
    from paper_2607_07862_b200 import build

    cuobjdump = "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not installed")
    sass = subprocess.run([cuobjdump, "-sass", build.build_lib()], capture_output=True, text=True).stdout
    lines = [l for l in sass.splitlines() if re.search(r"/\*[0-9a-f]{4,}\*/\s+\S", l)]
    mma = [i for i, l in enumerate(lines) if "UTCHMMA" in l]
    assert mma, "no tcgen05.mma in the library"
    for i in mma:
        window = " ".join(lines[i + 1:i + 4])
        assert "BRA.U.ANY" not in window, "UTCHMMA inside an elect loop:\n" + "\n".join(lines[i - 2:i + 4])


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "mlp_pipe.h"\nint main(void){ mlp_mode m = {0}; mlp_stats s; mlp_cta_record r; (void)m; (void)s; (void)r; '
                   'return (int)sizeof(mlp_mode) + (int)sizeof(mlp_stats) + (int)sizeof(mlp_cta_record); }\n')
    exe = tmp_path / "t"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    size = subprocess.run([str(exe)]).returncode
    from paper_2607_07862_b200 import binding as B

    assert size == (ctypes.sizeof(B.mlp_mode) + ctypes.sizeof(B.mlp_stats) + ctypes.sizeof(B.mlp_cta_record)) % 256


def test_struct_layouts_match_header_sizes(tmp_path):
    src = tmp_path / "s.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "mlp_pipe.h"\nint main(void){ printf("%zu %zu %zu %zu %zu %zu\\n", '
                   'sizeof(mlp_mode), sizeof(mlp_stats), sizeof(mlp_cta_record), offsetof(mlp_mode, split_k_layer), '
                   'offsetof(mlp_stats, runs), offsetof(mlp_cta_record, units)); return 0; }\n')
    exe = tmp_path / "s"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True).stdout.split()
    from paper_2607_07862_b200 import binding as B

    want = [ctypes.sizeof(B.mlp_mode), ctypes.sizeof(B.mlp_stats), ctypes.sizeof(B.mlp_cta_record),
            B.mlp_mode.split_k_layer.offset, B.mlp_stats.runs.offset, B.mlp_cta_record.units.offset]
    assert [int(x) for x in out] == want


def test_create_rejects_bad_arguments_without_a_gpu():
    """Argument validation happens before any CUDA call, so these hold on a CPU box too."""
    from paper_2607_07862_b200 import binding as B

    lib = B.load()
    h = ctypes.c_void_p()
    assert lib.mlp_pipe_create(None, 16, 64, 128, 128, 0, 0, None) == B.MLP_ERR_INVALID
    assert lib.mlp_pipe_create(ctypes.byref(h), 0, 64, 128, 128, 0, 0, None) == B.MLP_ERR_INVALID
    assert lib.mlp_pipe_create(ctypes.byref(h), 16, 60, 128, 128, 0, 0, None) == B.MLP_ERR_INVALID      # K % 8
    assert lib.mlp_pipe_create(ctypes.byref(h), 16, 64, 128, 128, 7, 0, None) == B.MLP_ERR_UNSUPPORTED  # dtype
    assert lib.mlp_pipe_create(ctypes.byref(h), 16, 64, 128, 128, 0, 9, None) == B.MLP_ERR_INVALID      # act
    bad = B.make_mode(B.MLP_MICROBATCH, chunks=3)
    assert lib.mlp_pipe_create(ctypes.byref(h), 16, 64, 128, 128, 0, 0, ctypes.byref(bad)) == B.MLP_ERR_INVALID
    bad = B.make_mode(B.MLP_CTA_PIPELINED, tile_m=24)
    assert lib.mlp_pipe_create(ctypes.byref(h), 16, 64, 128, 128, 0, 0, ctypes.byref(bad)) == B.MLP_ERR_INVALID
    bad = B.make_mode(B.MLP_CTA_PIPELINED, tile_m=512)
    assert lib.mlp_pipe_create(ctypes.byref(h), 16, 64, 128, 128, 0, 0, ctypes.byref(bad)) == B.MLP_ERR_UNSUPPORTED
    assert not h.value
    assert lib.mlp_pipe_last_error(None)
    assert lib.mlp_status_string(B.MLP_ERR_TIMEOUT) == b"flag-poll watchdog expired"
    assert lib.mlp_pipe_run(None, None, None, None, None, None) == B.MLP_ERR_INVALID
    lib.mlp_pipe_destroy(None)


def test_product_path_has_no_cpu_fallback_and_never_imports_the_oracle():
    import torch

    from paper_2607_07862_b200 import binding as B

    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            B.MlpPipe(16, [64, 128, 128], 0)
    pkg = os.path.join(ROOT, "paper_2607_07862_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "oracle_mlp" not in text, f
