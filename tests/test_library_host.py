"""-m "not gpu": the C-ABI library loads, exports every symbol include/genga_kick.h declares, and its
host-side logic (work decomposition, argument checks that need no device) behaves as documented.
No compute call is made here."""
import ctypes
import os
import re

import pytest

import paper_2201_10058_b200 as g

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2201_10058_b200 import build
    return build.build()


def test_every_declared_symbol_is_exported(built):
    header = open(os.path.join(ROOT, "include", "genga_kick.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(genga_kick\w*)\s*\(", header))
    assert declared, "no declarations found in include/genga_kick.h"
    lib = ctypes.CDLL(built)
    missing = [name for name in sorted(declared) if not hasattr(lib, name)]
    assert not missing, f"declared but not exported: {missing}"
    assert declared == set(g.EXPORTS), f"binding and header disagree: {declared ^ set(g.EXPORTS)}"


def test_every_declared_step_symbol_is_exported(built):
    header = open(os.path.join(ROOT, "include", "genga_step.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\bint\s+(genga_\w+)\s*\(", header))
    assert declared == set(g.STEP_EXPORTS), f"binding and header disagree: {declared ^ set(g.STEP_EXPORTS)}"
    lib = ctypes.CDLL(built)
    missing = [name for name in sorted(declared) if not hasattr(lib, name)]
    assert not missing, f"declared but not exported: {missing}"


def test_every_declared_group_symbol_is_exported(built):
    header = open(os.path.join(ROOT, "include", "genga_group.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\bint\s+(genga_\w+)\s*\(", header))
    assert declared == set(g.GROUP_EXPORTS)
    lib = ctypes.CDLL(built)
    assert all(hasattr(lib, name) for name in declared)


def test_every_declared_bs_symbol_is_exported(built):
    header = open(os.path.join(ROOT, "include", "genga_bs.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\bint\s+(genga_\w+)\s*\(", header))
    assert declared == set(g.BS_EXPORTS)
    lib = ctypes.CDLL(built)
    assert all(hasattr(lib, name) for name in declared)


def test_every_declared_senc_symbol_is_exported(built):
    header = open(os.path.join(ROOT, "include", "genga_senc.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\bint\s+(genga_\w+)\s*\(", header))
    assert declared == set(g.SENC_EXPORTS)
    lib = ctypes.CDLL(built)
    assert all(hasattr(lib, name) for name in declared)
    import ctypes as C
    assert C.sizeof(g.GengaSencConfig) == 40          # the struct of include/genga_senc.h: 4 x int32 + 3 x double


def test_strerror_texts(built):
    for code in (g.OK, g.E_NULL, g.E_ALIGN, g.E_SIZE, g.E_LEVEL, g.E_CUDA, g.E_NOMEM):
        assert g.strerror(code) and "unknown" not in g.strerror(code)
    assert "unknown" in g.strerror(-99)


def test_init_without_device_fails_loudly(built):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(g.GengaKickError) as e:
        g.GengaKick(128, 0)
    assert e.value.code == g.E_CUDA                  # no CPU fallback


def test_init_argument_checks(built):
    for nm, nt, lvl in [(-1, 0, 0), (0, 0, 0), (5, -2, 0)]:
        with pytest.raises(g.GengaKickError) as e:
            g.GengaKick(nm, nt, max_level=lvl)
        assert e.value.code == g.E_SIZE
    with pytest.raises(g.GengaKickError) as e:
        g.GengaKick(10, 0, max_level=-1)
    assert e.value.code == g.E_LEVEL


@pytest.mark.parametrize("nm,nt,level", [(1, 0, 0), (2048, 0, 0), (8192, 0, 0), (32770, 0, 1), (65536, 0, 0),
                                         (65536, 0, 1), (2048, 1048576, 0), (0, 500, 0), (257, 1, 0), (5000, 0, 2)])
def test_plan_covers_every_tile_once(built, nm, nt, level):
    sms = 148
    p = g.make_plan(nm, nt, level, sms)
    d = p.as_dict()
    assert d["i_block"] == d["threads"] * d["i_per_thread"]
    assert d["m_pad"] >= nm and d["m_pad"] % d["j_tile"] == 0
    n_i = d["m_pad"] + nt if nt else nm
    assert d["n_i_blocks"] * d["i_block"] >= n_i and d["n_rec"] >= n_i and d["n_rec"] % d["i_block"] == 0
    assert d["n_j_tiles"] * d["j_tile"] >= nm and d["n_tiles"] == d["n_i_blocks"] * d["n_j_tiles"]
    assert d["n_ctas"] <= max(d["n_tiles"], 0) or d["n_tiles"] == 0
    if d["n_tiles"] > d["n_ctas"]:
        assert d["n_ctas"] % sms == 0                # whole waves unless there are fewer tiles than that
    # ranges are contiguous, disjoint, cover [0, T), balanced to one tile
    prev, sizes, segs = 0, [], 1
    for c in range(d["n_ctas"]):
        t0, t1 = g.plan_cta_range(p, c)
        assert t0 == prev and t1 >= t0
        prev = t1
        sizes.append(t1 - t0)
        if t1 > t0:
            segs = max(segs, (t1 - 1) // d["n_j_tiles"] - t0 // d["n_j_tiles"] + 1)
    assert prev == d["n_tiles"]
    if sizes:
        assert max(sizes) - min(sizes) <= 1
    assert d["max_segs"] == segs
    assert d["partial_doubles"] == d["n_ctas"] * d["max_segs"] * 3 * d["i_block"]
    # the reduction pass visits exactly the CTAs whose range meets the i-block
    for ib in sorted({0, d["n_i_blocks"] // 2, d["n_i_blocks"] - 1}):
        if d["n_j_tiles"] == 0 or ib < 0:
            continue
        a, b = g.plan_iblock_ctas(p, ib)
        ta, tb = ib * d["n_j_tiles"], (ib + 1) * d["n_j_tiles"]
        meets = [c for c in range(d["n_ctas"]) if (lambda r: r[0] < tb and r[1] > ta and r[1] > r[0])(g.plan_cta_range(p, c))]
        assert meets == list(range(a, b + 1))


@pytest.mark.parametrize("nm,nt", [(2048, 1048576), (257, 1), (1, 100), (300, 5000), (16, 65520)])
def test_tp2_plan_covers_every_tile_once(built, nm, nt):
    """TP 2's second pass: massive bodies (i) x semi-active particles (j), same tile / CTA scheme."""
    sms = 148
    p = g.make_plan_tp2(nm, nt, sms)
    d, d0 = p.as_dict(), g.make_plan(nm, nt, 0, sms).as_dict()
    assert d["m_pad"] == d0["m_pad"] and d["n_rec"] == d0["n_rec"]
    assert d["n_i_blocks"] * d["i_block"] >= nm and d["n_i_blocks"] * d["i_block"] <= d["n_rec"]
    assert d["n_j_tiles"] * d["j_tile"] >= nt and d["m_pad"] + d["n_j_tiles"] * d["j_tile"] <= d["n_rec"]
    assert d["n_tiles"] == d["n_i_blocks"] * d["n_j_tiles"] and d["m_pad"] % 64 == 0
    prev, sizes = 0, []
    for c in range(d["n_ctas"]):
        t0, t1 = g.plan_cta_range(p, c)
        assert t0 == prev and t1 >= t0
        prev = t1
        sizes.append(t1 - t0)
    assert prev == d["n_tiles"] and max(sizes) - min(sizes) <= 1
    assert d["partial_doubles"] == d["n_ctas"] * d["max_segs"] * 3 * d["i_block"]


@pytest.mark.parametrize("nm,nt", [(65536, 0), (32770, 0), (24576, 0), (30001, 7), (65536, 1048576), (24575, 0), (100, 0)])
def test_symmetric_plan_covers_every_unordered_tile_once(built, nm, nt):
    """Level 0, massive x massive, every unordered pair once: rows of 1536-record i-blocks, row I holding the 256-record
    j-tiles jt >= 6 I, numbered row-major; CTA ranges contiguous, balanced under the cost model (a diagonal tile weighs
    1.4 symmetric tiles); the particles' rows one-sided beside it."""
    sms = 148
    p = g.make_plan_sym(nm, nt, sms)
    d = p.as_dict()
    IB = 1536
    assert d["symmetric"] == 1 and d["i_block"] == IB and d["j_tile"] == 256 and d["tiles_per_iblock"] == 6
    if nm < 24576:
        assert d["n_ctas"] == 0                       # the library keeps the one-sided kernel for small N
        return
    rows, njt, r = d["n_i_blocks"], d["n_j_tiles"], d["tiles_per_iblock"]
    assert rows * IB >= nm > (rows - 1) * IB and njt * 256 >= nm > (njt - 1) * 256
    # every (i-block, j-tile) with the j-tile at or beyond the i-block's first tile appears exactly once
    want = [(I, jt) for I in range(rows) for jt in range(I * r, njt)]
    assert d["n_tiles"] == len(want) and d["react_doubles"] == len(want) * 3 * 256
    for t in sorted({0, 1, len(want) // 3, len(want) // 2, len(want) - 2, len(want) - 1} | set(range(njt - 2, njt + 3))):
        I = g.plan_sym_row_of(p, t)
        assert (I, I * r + t - g.plan_sym_row_begin(p, I)) == want[t]
    assert g.plan_sym_row_begin(p, rows) == d["n_tiles"]
    # the unordered massive pairs are covered: tiles beyond the diagonal blocks + the diagonal blocks (one-sided there)
    assert d["n_ctas"] == sms
    import ctypes as C
    tab = (C.c_int64 * (sms + 1))()
    assert g.lib().genga_kick_plan_sym_table(C.byref(p), tab) == 0 and tab[0] == 0 and tab[sms] == d["n_tiles"]
    cost = lambda t: 14 if want[t][1] < (want[t][0] + 1) * r else 10          # diagonal : symmetric
    prev, costs, segs = 0, [], 1
    for c in range(d["n_ctas"]):
        t0, t1 = g.plan_cta_range(p, c)
        assert t0 == prev == tab[c] and t1 >= t0
        prev = t1
        costs.append(sum(cost(t) for t in range(t0, t1)))
        if t1 > t0:
            segs = max(segs, g.plan_sym_row_of(p, t1 - 1) - g.plan_sym_row_of(p, t0) + 1)
    assert prev == d["n_tiles"] and max(costs) - min(costs) <= 2 * 14             # balanced to a tile or two
    assert d["max_segs"] == segs and d["partial_doubles"] == sms * segs * 3 * IB
    for ib in sorted({0, rows // 2, rows - 1}):
        a, b = g.plan_iblock_ctas(p, ib)
        ta, tb = g.plan_sym_row_begin(p, ib), g.plan_sym_row_begin(p, ib + 1)
        meets = [c for c in range(d["n_ctas"]) if tab[c] < tb and tab[c + 1] > ta and tab[c + 1] > tab[c]]
        assert meets == list(range(a, b + 1))
    if nt:
        q = g.make_plan_tprows(nm, nt, sms).as_dict()
        assert q["symmetric"] == 0 and q["m_pad"] == d["m_pad"] and q["n_i_blocks"] * q["i_block"] >= nt
        assert q["n_j_tiles"] * q["j_tile"] >= nm and q["n_tiles"] == q["n_i_blocks"] * q["n_j_tiles"]
        assert q["m_pad"] + q["n_i_blocks"] * q["i_block"] <= q["n_rec"]


def test_plan_errors(built):
    with pytest.raises(g.GengaKickError) as e:
        g.make_plan(0, 0, 0, 148)
    assert e.value.code == g.E_SIZE
    with pytest.raises(g.GengaKickError) as e:
        g.make_plan(10, 0, -1, 148)
    assert e.value.code == g.E_LEVEL
    with pytest.raises(g.GengaKickError) as e:
        g.make_plan(10, 0, 0, 0)
    assert e.value.code == g.E_SIZE


def test_product_does_not_touch_the_oracle():
    """The product path may not import, link or read oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2201_10058_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
                assert "oracle/" not in text.replace("shared with oracle/", "").replace("imports oracle/", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2201_10058_b200" not in text.replace("paper_2201_10058_b200/csrc/", "") or f.endswith(".c")
            assert not re.search(r"^\s*(from|import)\s+paper_2201_10058_b200\b", text, flags=re.M), f
