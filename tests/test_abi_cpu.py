"""CPU-only checks of the boundary: libctr.so loads and exports every symbol include/ctr.h
declares; the ctypes structs match the header field for field; the product has no CPU fallback."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
HEADER = (ROOT / "include" / "ctr.h").read_text()


@pytest.fixture(scope="module")
def lib():
    from paper_1009_2288_b200 import build as ctr_build
    ctr_build.build()
    import paper_1009_2288_b200 as ctr
    return ctr.load_library()


def declared_functions():
    body = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    return sorted(set(re.findall(r"\b(ctr_[a-z_0-9]+)\s*\(", body)))


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert {"ctr_create", "ctr_destroy", "ctr_forward", "ctr_back", "ctr_cgls", "ctr_update_weights",
            "ctr_eptv_step", "ctr_reconstruct", "ctr_set_params", "ctr_get_stats", "ctr_strerror",
            "ctr_last_error"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/ctr.h but not exported by libctr.so"


def test_binding_lists_every_header_function():
    import paper_1009_2288_b200 as ctr
    assert sorted(ctr.EXPORTS) == declared_functions()


def _struct_fields(name):
    clean = re.sub(r"/\*.*?\*/", "", HEADER, flags=re.S)
    m = re.search(r"typedef struct \{([^{}]*)\}\s*" + name + ";", clean)
    body = m.group(1)
    out = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        toks = re.match(r"(const\s+float\s*\*|int32_t|float|double)\s*(.*)", decl, flags=re.S)
        kind = toks.group(1).replace(" ", "")
        for nm in toks.group(2).split(","):
            out.append((nm.strip(), kind))
    return out


def test_ctypes_structs_match_header():
    import paper_1009_2288_b200 as ctr
    kinds = {"int32_t": C.c_int32, "float": C.c_float, "double": C.c_double, "constfloat*": C.POINTER(C.c_float)}
    for name, struct in (("ctr_geometry", ctr.ctr_geometry), ("ctr_params", ctr.ctr_params),
                         ("ctr_sweep_stat", ctr.ctr_sweep_stat), ("ctr_peaks", ctr.ctr_peaks)):
        hdr = _struct_fields(name)
        got = [(n, t) for n, t in struct._fields_]
        assert len(hdr) == len(got), name
        for (hn, hk), (gn, gt) in zip(hdr, got):
            assert gt is kinds[hk] or gt == kinds[hk], (name, hn, gn)
            assert hn == gn or (hn, gn) == ("lambda", "lam"), (name, hn, gn)


def test_strerror_and_defaults_without_a_gpu(lib):
    import paper_1009_2288_b200 as ctr
    assert lib.ctr_strerror(0) == b"ok"
    assert b"invalid" in lib.ctr_strerror(-1)
    p = ctr.make_params()
    assert (p.n_gd, p.armijo_max, p.positivity) == (5, 16, 1)
    assert abs(p.sigma_quantile - 0.9) < 1e-6 and abs(p.armijo_t0 - 1e-3) < 1e-9


def test_null_arguments_are_rejected_without_touching_cuda(lib):
    h = C.c_void_p()
    assert lib.ctr_create(None, C.byref(h)) == -1 and not h.value
    assert lib.ctr_forward(None, None, None, None) == -1
    assert lib.ctr_set_params(None, None) == -1
    lib.ctr_destroy(None)


def test_product_never_imports_the_oracle():
    """The CUDA path and its binding must not reference oracle/ (no CPU fallback)."""
    pkg = ROOT / "paper_1009_2288_b200"
    for f in list(pkg.glob("*.py")) + list((pkg / "csrc").glob("*")):
        txt = f.read_text()
        assert "import oracle" not in txt and "from oracle" not in txt and "ctr_oracle" not in txt, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c"):
            assert "paper_1009_2288_b200 import" not in f.read_text() and "libctr.so" not in f.read_text(), f


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    import paper_1009_2288_b200.binding as b
    monkeypatch.setattr(b, "_lib", None)
    monkeypatch.setattr(b, "_LIB_PATH", tmp_path / "libctr.so")
    with pytest.raises(FileNotFoundError):
        b.load_library()
