"""Host logic behind the device image of a cloud (csrc/pdv_api.cu::build_blob), checked on the CPU (no GPU needed) against the
definitions the ORACLE's tables give: the class pick through the class guide and the two threshold tables, the depth probe
through the depth guide and the one-probe rows, the phase rows.  The test reads the image through pdv_cloud_get_image and walks
it the way include/pdv.h / csrc/pdv_device.h say it is to be read; the expected values come from oracle/cloud.py.

These are the invariants the flight loop relies on without checking: a wrong guide entry is a wrong class or an out-of-range
table index on the device."""
import math

import numpy as np
import pytest

import pdv_workloads as W
from oracle import cloud as ocloud

pytestmark = pytest.mark.usefixtures("_library_is_built")

LN2 = math.log(2.0)


@pytest.fixture(scope="module")
def P():
    import paper_2012_00963_b200 as P
    return P


CLOUDS = {
    "cfg2_mono": lambda: W.config(1)["clouds"][0],
    "cfg3_poly": lambda: W.config(2)["clouds"][0],
    "cfg5_poly_tiny_classes": lambda: W.config(4)["clouds"][0],
    "thick_mono": lambda: W._cloud(20.0, 6.0, 2000.0, diameter_um=1.0),
    "paper_base": lambda: W.paper_base_case()["clouds"][0],
    "three_classes": lambda: dict(W.config(1)["clouds"][0], diameters=[0.15e-6, 0.4e-6, 5e-6], number_weights=[0.6, 0.3, 0.1]),
}


def _pick_from_image(img, cw, table):
    """Class of class word `cw` read from the image: guide byte, one compare, walk in flagged cells (pdv_device.h)."""
    L = img["layout"]
    e = int(img["cguide"][cw >> L["cguide_shift"]])
    thr = img[table]
    c = e & 0x7F
    if int(thr[c]) <= cw:
        c += 1
    if e & 0x80:
        while c < L["n_classes"] - 1 and int(thr[c]) <= cw:
            c += 1
    return c, e


def _class_by_definition(p_class, cw):
    """DESIGN.md D2: c = #{j < n-1 : (cw + 1/2) / 2^32 >= cum_j}."""
    cum = np.cumsum(np.asarray(p_class, dtype=np.float64))[:-1]
    return int(np.sum((cw + 0.5) / 4294967296.0 >= cum))


@pytest.mark.parametrize("name", list(CLOUDS))
def test_class_pick_through_guide_and_thresholds(P, name):
    params = CLOUDS[name]()
    oc = ocloud.build_cloud(params)
    img = P.pdv_cloud_create(params).image()
    L = img["layout"]
    n = L["n_classes"]
    assert n == len(oc.p_class)
    assert L["cguide_cells"] == 1 << (32 - L["cguide_shift"]) and img["cguide"].size == L["cguide_cells"]
    assert L["off_cguide"] + L["cguide_cells"] <= L["image_bytes"]
    # every guide entry is a valid class count; the flag count is what the header says
    assert int((img["cguide"] & 0x7F).max()) <= max(n - 2, 0)
    assert int((img["cguide"] >> 7).sum()) == L["cguide_flagged"]
    rng = np.random.default_rng(5)
    words = set(int(x) for x in rng.integers(0, 1 << 32, size=4000, dtype=np.uint64))
    words |= {0, 1, 127, 128, 129, 255, 256, 0xFFFFFFFF, 0xFFFFFFFE, 0xFFFFFF80, 0xFFFFFF7F, 0x80000000}
    thr = [int(t) for t in img["thr"][:max(n - 1, 0)]]
    for t in thr:                                            # around every threshold, and around its cell and byte borders
        for d in (-257, -256, -129, -128, -127, -2, -1, 0, 1, 2, 127, 128, 129, 255, 256):
            words.add(min(max(t + d, 0), 0xFFFFFFFF))
        words.add(t & ~((1 << L["cguide_shift"]) - 1))
        words.add(min((t | ((1 << L["cguide_shift"]) - 1)), 0xFFFFFFFF))
    for cw in sorted(words):
        want = _class_by_definition(oc.p_class, cw) if n > 1 else 0
        got, e = _pick_from_image(img, cw, "thr")
        if n == 1:
            assert e == 0 and got <= 1                       # one class: "class 1" (word 0xffffffff only) is the stored copy of class 0
            continue
        assert got == want, (hex(cw), got, want)
        assert L["cguide_flagged"] or not (e & 0x80)
        # first / second flight of a group: the RAW word against thr24 == the masked word against thr
        masked = (cw & 0xFFFFFF00) | 0x80
        got24, _ = _pick_from_image(img, cw, "thr24")
        assert got24 == _class_by_definition(oc.p_class, masked), (hex(cw), got24)
    if n > 1:                                                # thresholds are the oracle's cumulative probabilities
        cum = np.cumsum(oc.p_class)[:-1]
        assert np.all(np.abs(np.asarray(thr, dtype=np.float64) - (cum * 4294967296.0 - 0.5)) <= 1.0)
        assert np.all(img["thr"][n - 1:] == 0xFFFFFFFF)
        assert np.allclose(img["albedo"][:n], np.asarray(oc.omega0), rtol=0, atol=1e-7)
    else:
        assert img["albedo"][0] == img["albedo"][1] and np.array_equal(img["phase"][0], img["phase"][1])


def test_clean_and_flagged_guides_are_what_the_design_says(P):
    assert P.pdv_cloud_create(CLOUDS["cfg3_poly"]()).image()["layout"]["cguide_flagged"] == 0          # -> the ALT instantiation
    lay = P.pdv_cloud_create(CLOUDS["cfg5_poly_tiny_classes"]()).image()["layout"]
    assert lay["cguide_flagged"] == 1 and lay["cguide_shift"] == 20                                    # one cell in 4096 walks


@pytest.mark.parametrize("name", list(CLOUDS))
def test_depth_probe_through_guide_and_rows(P, name):
    """One guide load + one row: for every optical depth T of the cloud the probe must return the velocity of the oracle's
    canonical depth table (bins uniform in v, T linear in v inside a bin, R24) -- in units of ln 2 on the device."""
    params = CLOUDS[name]()
    oc = ocloud.build_cloud(params)
    img = P.pdv_cloud_create(params).image()
    L = img["layout"]
    nd = L["n_depth_bins"]
    assert L["depth_bisect"] == 0
    T_edge = np.asarray(oc.T_edge, dtype=np.float64)          # T_0 = 0 (top) ... T_nd = tau_ext, oracle units
    v_edge = oc.v_max - np.arange(nd + 1) * (oc.v_max - oc.v_fs) / nd          # bins uniform in v, j = 0 at the top (R24)
    assert img["rows"][:, 0] == pytest.approx(T_edge[1:] / LN2, rel=2e-7)
    assert L["tau_ext_ln2"] == pytest.approx(oc.tau_ext / LN2, rel=2e-7)
    assert img["rows"][:, 1] == pytest.approx(0.5 * v_edge[1:], rel=2e-7)
    assert L["off_rows"] - L["off_phase"] >= 8 * max(L["n_classes"], 2) * L["n_phase_bins"] + 80       # room for the round keys
    rng = np.random.default_rng(7)
    tau = float(np.float32(L["tau_ext_ln2"]))
    Ts = np.concatenate([rng.uniform(0.0, tau, 3000), tau * rng.uniform(0, 1, 2000) ** 6, img["rows"][:, 0].astype(np.float64),
                         np.nextafter(img["rows"][:, 0], np.float32(0)).astype(np.float64), [tau, 1e-30, 1e-12]])
    Ts = np.minimum(Ts, tau).astype(np.float32)
    Ts = Ts[Ts > 0]
    bits = Ts.view(np.uint32)
    cell = np.maximum(bits >> L["guide_shift"], L["guide_base"]) - L["guide_base"]
    assert int(cell.max()) < L["n_guide"]
    j = img["guide"][cell].astype(np.int64)
    assert int(j.max()) < nd
    x = img["rows"][j]
    # the row's edge T_{j+1} and the edge before / after it bracket T:  T_j <= T < T_{j+2}
    Tf = np.concatenate([[0.0], img["rows"][:, 0].astype(np.float64), [np.inf]])
    assert np.all(Tf[j] <= Ts) and np.all(Ts < Tf[j + 2] + (Tf[j + 2] == tau) * 1.0)
    slope = np.where(Ts < x[:, 0], x[:, 2], x[:, 3])
    vh = x[:, 1] + (Ts - x[:, 0]).astype(np.float32) * slope
    want = 0.5 * np.interp(Ts.astype(np.float64) * LN2, T_edge, v_edge)
    # fp32 tables: the probe reproduces the canonical table to a few 1e-7 of v (plus the slope times the fp32 spacing of T)
    tol = 4e-7 * want + np.abs(slope) * np.spacing(Ts) * 2 + 1e-3
    assert np.all(np.abs(vh - want) <= tol), float(np.max(np.abs(vh - want) / want))


def test_phase_rows_are_the_oracle_table(P):
    params = CLOUDS["cfg3_poly"]()
    oc = ocloud.build_cloud(params)
    img = P.pdv_cloud_create(params).image()
    L = img["layout"]
    K = L["n_phase_bins"]
    M = np.asarray(oc.phase, dtype=np.float64).reshape(L["n_classes"], K + 1)
    assert img["phase"][:L["n_classes"], :, 0] == pytest.approx(M[:, :-1], abs=2e-7)
    shiftK = 32 - L["log2_phase_bins"]
    assert img["phase"][:L["n_classes"], :, 1] * 2.0 ** shiftK == pytest.approx(np.diff(M, axis=1), abs=3e-7)
    assert L["frac_mask"] == 0xFFF << (shiftK - 12)
