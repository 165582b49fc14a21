"""The C-ABI library loads and exports every symbol include/b200_allegro.h declares (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "b200_allegro.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(allegro_[a-z0-9_]+)\s*\(", src)) - {"allegro_alloc_fn", "allegro_free_fn"})


def test_library_builds_loads_and_exports_all_symbols():
    import paper_2304_10061_b200 as P
    P.build_library()
    lib = P.load_library()
    names = _declared()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(P.EXPORTS)


def test_host_logic_without_gpu():
    import paper_2304_10061_b200 as P
    from synthetic import CONFIGS
    from synthetic.weights import blob_num_floats
    lib = P.load_library()
    for cfg, want_paths, want_dims in [(CONFIGS[0], [2], [4, 1]), (CONFIGS[1], [11, 3], [9, 9, 1]),
                                       (CONFIGS[4], [34, 34, 4], [16, 31, 16, 1])]:
        hp = P.hparams_from(cfg.hp)
        fan = P.path_fan(hp)
        assert [len(f) for f in fan] == want_paths
        assert P.layer_dims(hp) == want_dims
        nbytes = ctypes.c_size_t(0)
        assert lib.allegro_blob_size(ctypes.byref(hp), ctypes.byref(nbytes)) == 0
        nfl = blob_num_floats(cfg.hp, want_paths)
        assert nbytes.value == nfl * 4 + (nfl * 4) % 8 + 16 * cfg.hp.n_species
    # error behaviour: bad hyper-parameters, bad blob size
    hp = P.hparams_from(CONFIGS[0].hp)
    hp.l_max = 7
    assert lib.allegro_blob_size(ctypes.byref(hp), ctypes.byref(nbytes)) == -1
    assert b"l_max" in lib.allegro_last_error(None)
    hp = P.hparams_from(CONFIGS[0].hp)
    h = ctypes.c_void_p(None)
    buf = ctypes.create_string_buffer(100)
    assert lib.allegro_create(ctypes.byref(hp), buf, 100, ctypes.byref(h)) == -2


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2304_10061_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h", ".cuh")):
                txt = open(os.path.join(dp, f)).read()
                assert "oracle" not in txt.replace("oracle/ (no shared code)", ""), (f, "product code must not reference oracle/")
    for f in ("oracle/allegro_oracle.py",):
        txt = open(os.path.join(ROOT, f)).read()
        assert "import paper_2304_10061_b200" not in txt and "from paper_2304_10061_b200" not in txt


def test_16bit_operand_modes_check_their_preconditions():
    """Precision 2 / 4 (bf16 / fp16 operand MLPs) are real modes with shape preconditions (include/b200_allegro.h); a model
    that does not meet them is refused with ALLEGRO_ERR_BAD_HPARAMS instead of silently running another mode.  The
    hyper-parameter check runs before any device is touched, so this needs no GPU."""
    import ctypes as C
    import dataclasses
    import paper_2304_10061_b200 as P
    from synthetic import CONFIGS
    lib = P.load_library()
    n = C.c_size_t(0)
    for prec in (2, 4):
        ok = P.hparams_from(CONFIGS[1].hp, prec)
        assert lib.allegro_blob_size(C.byref(ok), C.byref(n)) == 0 and n.value > 0
        one_layer = P.hparams_from(dataclasses.replace(CONFIGS[1].hp, twobody_dims=(256,)), prec)
        assert lib.allegro_blob_size(C.byref(one_layer), C.byref(n)) == -1
        odd_latent = P.hparams_from(dataclasses.replace(CONFIGS[1].hp, latent_dims=(96, 256)), prec)
        assert lib.allegro_blob_size(C.byref(odd_latent), C.byref(n)) == -1
        assert b"16-bit" in lib.allegro_last_error(None)
    bad = P.hparams_from(CONFIGS[1].hp, 5)
    assert lib.allegro_blob_size(C.byref(bad), C.byref(n)) == -1
