"""The C-ABI boundary without a GPU: liblsp_b200.so builds (nvcc cross-compiles sm_100a), loads, exports every
symbol include/lsp.h declares, validates arguments on the host, and fails loudly -- LSP_ERR_CUDA, never a CPU
fallback -- when no device is present.  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lsp.h")


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # drop comments
    names = re.findall(r"\b(lsp_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def pkg():
    import paper_2105_04006_b200 as p
    p.load_library()
    return p


def test_header_declares_the_four_calls():
    names = declared_functions()
    for required in ("lsp_plan_create", "lsp_periodogram_batched", "lsp_best_period", "lsp_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(pkg):
    lib = pkg.load_library()
    names = declared_functions()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"liblsp_b200.so does not export {n}"
    # and the binding's own list is the header's list
    assert sorted(pkg.EXPORTS) == names


def test_no_torch_or_cxx_types_in_header():
    src = open(HEADER).read()
    code = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    for bad in ("torch", "at::", "std::", "template", "class ", "cudaStream_t"):
        assert bad not in code
    assert 'extern "C"' in code


def test_config_struct_layout_matches_header(pkg):
    # 2 doubles + int64 + 6 int32 + 3 int64 + 2 int32 + int64 + 4 int32 = 8*3 + 4*6 + 8*3 + 4*2 + 8 + 4*4 = 104 bytes, no padding
    assert ctypes.sizeof(pkg.LspConfig) == 104
    assert pkg.LspConfig.n_freq.offset == 16 and pkg.LspConfig.chunk_bytes.offset == 48 and pkg.LspConfig.kernel.offset == 72
    assert pkg.LspConfig.flags.offset == 76 and pkg.LspConfig.table_budget_bytes.offset == 80
    assert pkg.LspConfig.tensor_roles.offset == 88 and pkg.LspConfig.tensor_b_stages.offset == 92
    assert pkg.LspConfig.tensor_products.offset == 96 and pkg.LspConfig.tensor_pair.offset == 100
    # the header's struct has the same fields in the same order
    src = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    body = re.search(r"typedef struct lsp_config \{(.*?)\} lsp_config;", src, flags=re.S).group(1)
    fields = re.findall(r"\b(?:double|int64_t|int32_t)\s+([a-z_0-9]+)\s*;", body)
    assert fields == [f[0] for f in pkg.LspConfig._fields_]


def test_library_is_built_for_sm_100a_only():
    from paper_2105_04006_b200 import build
    assert "arch=compute_100a,code=sm_100a" in " ".join(build.NVCC_FLAGS) and "-lineinfo" in build.NVCC_FLAGS
    log = open(os.path.join(os.path.dirname(build.LIB), "build.log")).read() if os.path.exists(
        os.path.join(os.path.dirname(build.LIB), "build.log")) else ""
    if log:
        assert "sm_100a" in log


@pytest.mark.parametrize("kw", [dict(f_min=0.0), dict(f_min=-1.0), dict(f_max=0.05), dict(n_freq=0),
                                dict(dtype=1, fast_math=1), dict(dtype=7), dict(kernel=9), dict(flags=2),
                                dict(n_copy_streams=99), dict(table_budget_bytes=-1), dict(tensor_roles=3),
                                dict(tensor_b_stages=1), dict(tensor_b_stages=9), dict(tensor_products=1),
                                dict(tensor_products=4), dict(tensor_pair=3), dict(tensor_pair=-1)])
def test_plan_create_rejects_bad_arguments_on_host(pkg, kw):
    args = dict(f_min=0.1, f_max=2.0, n_freq=10, dtype=0, fast_math=0, normalize=0, center=0, device=0,
                n_copy_streams=0, chunk_bytes=0, max_objects=0, max_total_obs=0, kernel=0, flags=0,
                table_budget_bytes=0, tensor_roles=0, tensor_b_stages=0, tensor_products=0, tensor_pair=0)
    args.update(kw)
    cfg = pkg.LspConfig(**args)
    with pytest.raises(pkg.LspError) as ei:
        pkg.lsp_plan_create(cfg)
    assert ei.value.status == 1        # LSP_ERR_INVALID_ARG, decided before any CUDA call


def test_no_cpu_fallback_without_a_device(pkg):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is visible")
    cfg = pkg.LspConfig(0.1, 2.0, 10, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0)
    with pytest.raises(pkg.LspError) as ei:
        pkg.lsp_plan_create(cfg)
    assert ei.value.status == 2        # LSP_ERR_CUDA
    assert "no CPU fallback" in str(ei.value)


def test_null_plan_calls_are_safe(pkg):
    lib = pkg.load_library()
    lib.lsp_destroy(None)
    assert lib.lsp_best_period(None, 0, None, None, None, None, None, None, None, None) == 1
    assert lib.lsp_periodogram_batched_host(None, 0, None, None, None, None, None, None, None, None) == 1
    assert lib.lsp_best_merge(None, 0, 1, None, None, None, None, None, None) == 1
    assert isinstance(pkg.lsp_version(), str) and "sm_100a" in pkg.lsp_version()


def test_product_path_never_touches_the_oracle():
    """The package (product path) must not import, read or run anything under oracle/ or _work/."""
    pkg_dir = os.path.join(ROOT, "paper_2105_04006_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "lsp_oracle" not in text, f
                assert "_work" not in text, f


def test_library_reads_no_environment_variables():
    """Behaviour is switched through lsp_config only: no getenv in the library or its binding."""
    pkg_dir = os.path.join(ROOT, "paper_2105_04006_b200")
    for dirpath, _, files in os.walk(pkg_dir):
        for f in files:
            if f.endswith((".cu", ".cuh")) or f == "binding.py":
                text = open(os.path.join(dirpath, f)).read()
                assert "getenv" not in text and "os.environ" not in text, f
