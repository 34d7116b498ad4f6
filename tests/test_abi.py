"""The C-ABI shared library loads without a GPU and exports every symbol include/jefi.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "jefi.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(jefi_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_six_calls():
    syms = declared_symbols()
    for name in ("jefi_create", "jefi_push_sources", "jefi_field_step", "jefi_deposit", "jefi_push_particles", "jefi_destroy"):
        assert name in syms


def test_library_exports_every_declared_symbol():
    from paper_2209_07944_b200 import build, jefi

    build.build_lib()
    lib = ctypes.CDLL(jefi.LIB_PATH)
    for name in declared_symbols():
        assert hasattr(lib, name), name
    assert sorted(jefi.EXPORTS) == declared_symbols()  # the binding wraps exactly the declared calls


def test_create_rejects_bad_arguments_without_a_gpu():
    """Argument validation happens before any CUDA call, so these error codes are testable on a CPU box."""
    from paper_2209_07944_b200 import jefi

    lib = jefi.load_library()
    h = ctypes.c_void_p()
    assert lib.jefi_create(None, ctypes.byref(h)) == jefi.JEFI_EINVAL
    cfg = jefi.jefi_config(0, 4, 4, 1e-4, 1e-4, 1e-4, 1e-13)
    assert lib.jefi_create(ctypes.byref(cfg), ctypes.byref(h)) == jefi.JEFI_EINVAL and not h.value
    assert b"positive" in lib.jefi_last_error(None)
    lib.jefi_destroy(None)


def test_config_init_checks_the_struct_size_and_zeroes_it():
    """jefi_config has no version member: jefi_config_init(cfg, sizeof) refuses a struct of another size (a caller built against an
    older header) and otherwise fills in the all-zero defaults.  No GPU needed."""
    from paper_2209_07944_b200 import jefi

    lib = jefi.load_library()
    cfg = jefi.jefi_config(5, 6, 7, 1.0, 2.0, 3.0, 4.0)
    cfg.field_tile = 99
    assert lib.jefi_config_init(ctypes.byref(cfg), ctypes.sizeof(jefi.jefi_config) - 12) == jefi.JEFI_EINVAL
    assert b"rebuild" in lib.jefi_last_error(None) and cfg.nx == 5 and cfg.field_tile == 99  # untouched
    assert lib.jefi_config_init(None, ctypes.sizeof(jefi.jefi_config)) == jefi.JEFI_EINVAL
    assert lib.jefi_config_init(ctypes.byref(cfg), ctypes.sizeof(jefi.jefi_config)) == jefi.JEFI_OK
    assert bytes(cfg) == bytes(ctypes.sizeof(jefi.jefi_config))
    # the binding's mirror of the struct matches the header member for member (same count, same order)
    text = open(os.path.join(ROOT, "include", "jefi.h")).read()
    body = re.sub(r"/\*.*?\*/", "", text[text.index("typedef struct {"):text.index("} jefi_config;")], flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if decl:
            names += [re.sub(r"\[.*\]", "", n).strip(" *") for n in decl.split(None, 1)[1].split(",")]
    assert names == [f[0] for f in jefi.jefi_config._fields_], names


def test_product_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package, bench's product arm or include/ may name it."""
    pkg = os.path.join(ROOT, "paper_2209_07944_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "jefi_oracle" not in src, f
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for f in files:
            if f.endswith((".py", ".c", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+paper_2209_07944_b200", src, flags=re.M), f


def test_bench_traffic_table_belongs_to_this_kernel_source():
    """bench.py's roofline.traffic comes from a committed ncu capture and is valid only for the kernel source it was taken from
    (sha1 of csrc/jefi_field.cu + csrc/jefi_ctx.h): the table must name the current source and an existing profiles/ file."""
    import os
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    sys.path.insert(0, root)
    import bench

    nbytes, prof = bench.field_traffic("cfg4_96c_field_only", "nearest")
    assert nbytes is not None and nbytes > 4.74e9, prof  # at least one pass over the ring's S half
    assert os.path.exists(os.path.join(root, prof)), prof
    assert bench.kernel_source_sha() in open(os.path.join(root, prof)).read()
