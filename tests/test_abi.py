"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/chfpe.h declares; descriptor validation and workspace sizing run on the CPU."""
import ctypes as C
import os
import re

import pytest

import chfpe_inputs as ci

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_functions():
    text = open(os.path.join(ROOT, "include", "chfpe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(chfpe_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    import paper_2509_25840_b200 as P
    L = P.lib()
    names = header_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), "libchfpe.so does not export %s" % n
    assert sorted(P.EXPORTED_SYMBOLS) == names


def test_oracle_and_product_share_no_code():
    """The oracle never imports the product and vice versa; the product never touches oracle/."""
    for sub, banned in (("oracle", "paper_2509_25840_b200"), ("paper_2509_25840_b200", "oracle")):
        for dirpath, _, files in os.walk(os.path.join(ROOT, sub)):
            for f in files:
                if f.endswith((".py", ".c", ".h", ".cu", ".cuh")):
                    src = open(os.path.join(dirpath, f)).read()
                    assert ("import " + banned) not in src and ("from " + banned) not in src
                    if sub == "paper_2509_25840_b200":
                        assert "chfpe_ref" not in src


def test_workspace_bytes_and_validation():
    import paper_2509_25840_b200 as P
    for name, arrays in (("cfg1", 4), ("cfg4", 4)):
        cfg = ci.config(name)
        K = {"cfg1": 9, "cfg4": 20}[name]
        cells = 1
        for s in range(cfg["n_modes"]):
            cells *= cfg["nq"][s] * cfg["np"][s]
        nbytes = P.workspace_bytes(cfg, batch=1)
        assert arrays * K * cells * 8 <= nbytes <= arrays * K * cells * 8 + (8 << 20)
    n5 = P.workspace_bytes(ci.config("cfg5"), batch=5)
    assert n5 < 180e9                       # config 5 with 5 slots (trajectory + 4 replicas) fits one B200
    for bad in (dict(nq=[4]), dict(depth=-1), dict(beta=0.0), dict(gamma=[0.0]), dict(U=[(1.0, (5,))]),
                dict(scheme="compact6", nq=[5000])):
        with pytest.raises(P.ChfpeError):
            P.workspace_bytes(ci.config("cfg1", **bad))
    with pytest.raises(P.ChfpeError):
        P.workspace_bytes(ci.config("cfg1"), batch=0)
    # COMPACT6 (step a9) needs three element-sized scratch arrays on top of the explicit schemes' workspace
    extra = P.workspace_bytes(ci.config("cfg1", scheme="compact6")) - P.workspace_bytes(ci.config("cfg1"))
    assert 3 * 64 * 64 * 8 <= extra <= 3 * 64 * 64 * 8 + (1 << 20)


def test_create_rejects_bad_workspace_without_touching_the_gpu():
    import paper_2509_25840_b200 as P
    from paper_2509_25840_b200 import binding
    d, keep = binding.make_desc(ci.config("cfg1"))
    h = C.c_void_p()
    rc = P.lib().chfpe_create(C.byref(d), None, 0, None, C.byref(h))
    assert rc == -2 and not h.value          # CHFPE_ERR_WORKSPACE


def test_hermite_workspace_bytes_and_validation():
    """Row f1 host logic without a GPU: workspace sizing (three state-sized arrays per slot + tables) and descriptor
    validation of the chfpe_hermite_* entry points; create refuses a missing workspace before touching CUDA."""
    import paper_2509_25840_b200 as P
    from paper_2509_25840_b200 import binding
    cfg = ci.config("cfg4h")
    values = 20 * 8 ** 3 * 32 ** 3
    for batch in (1, 3):
        n = P.hermite_workspace_bytes(cfg, batch=batch)
        assert 3 * batch * values * 8 <= n <= 3 * batch * values * 8 + (16 << 20)
    assert P.hermite_workspace_bytes(ci.config("cfg4h", scheme="compact6")) >= 3 * values * 8
    for bad in (dict(nq=[4, 32, 32]), dict(np=[0, 8, 8]), dict(depth=-1), dict(beta=0.0), dict(gamma=[0.0, 1.0, 1.0]),
                dict(scheme="compact6", nq=[300, 32, 32])):
        with pytest.raises(P.ChfpeError):
            P.hermite_workspace_bytes(ci.config("cfg4h", **bad))
    with pytest.raises(P.ChfpeError):
        P.hermite_workspace_bytes(cfg, batch=0)
    d, keep = binding.make_desc(binding._hermite_cfg(ci.config("cfg2", nq=[64], np=[8])))
    h = C.c_void_p()
    rc = P.lib().chfpe_hermite_create(C.byref(d), None, 0, None, C.byref(h))
    assert rc == -2 and not h.value          # CHFPE_ERR_WORKSPACE


def test_every_environment_knob_is_documented_in_the_header():
    """include/chfpe.h ("Tunables") lists every CHFPE_* environment variable the library reads (kernel variants and launch
    plans that compute the same results): a knob added to csrc/ without a line there fails this test."""
    import glob
    import re
    root = os.path.join(os.path.dirname(__file__), "..")
    names = set()
    for f in glob.glob(os.path.join(root, "paper_2509_25840_b200", "csrc", "*")):
        names |= set(re.findall(r'(?:getenv|env_int)\("(CHFPE_[A-Z0-9_]+)"', open(f).read()))
    assert len(names) >= 20
    header = open(os.path.join(root, "include", "chfpe.h")).read()
    missing = sorted(n for n in names if n not in header)
    assert not missing, missing

