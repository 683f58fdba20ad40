"""CPU tests of the boundary: the C-ABI library loads, exports every symbol include/jerk.h declares,
and its host-only logic (plan geometry, validation, sizes) agrees with the oracle's definitions.
No compute call is made here (no GPU)."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

from oracle import jerk_oracle as orc
from paper_1911_01353_b200 import binding, build
import workloads as synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load_library()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "jerk.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(jerk_[a-z_]+)\s*\(", hdr))
    assert names == set(binding.EXPORTS), names ^ set(binding.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_cand_record_is_16_bytes():
    assert binding.CAND_DTYPE.itemsize == 16


@pytest.mark.parametrize("idx", [1, 2, 3, 4])
def test_plan_geometry_matches_survey_table(lib, idx):
    cfg = synth.config(idx)
    p = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    want = {1: (21, 7, 33, 958, 25), 2: (101, 31, 133, 1782, 125), 3: (201, 61, 258, 3580, 250), 4: (201, 61, 258, 7676, 250)}[idx]
    i = p.info
    assert (i.nz, i.nw, i.hw_max, i.step, i.c_max) == want          # SURVEY.md 8(a) size table
    assert i.points == 2 * cfg.nbins * i.nz * i.nw
    assert i.seg_base % 2 == 0 and i.seg_base <= -(i.c_max + i.hw_max)
    # coverage: first segment reaches b <= 0 for c = -c_max.., last reaches nbins-1 for c = +c_max
    assert i.seg_base + i.hw_max + i.c_max <= 0
    assert i.seg_base + (i.nseg - 1) * i.step + i.hw_max + i.step - 1 - i.c_max >= cfg.nbins - 1
    assert i.bank_bytes >= i.ntemplates * 2 * cfg.seg_len * 8
    flops_unit = 5 * cfg.seg_len * math.log2(cfg.seg_len) + 6 * cfg.seg_len + 3 * i.step
    assert abs(i.flops_per_search - math.ceil(cfg.nbins / i.step) * 2 * i.ntemplates * flops_unit) < 1e-6 * i.flops_per_search


def test_template_geometry_matches_oracle(lib):
    cfg = synth.config(3)
    p = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    for iw in range(p.info.nw):
        for iz in range(0, p.info.nz, 1):
            c, hw = p.template_geometry(iz, iw)
            assert c == orc.centre(float(zs[iz]), float(ws[iw])), (zs[iz], ws[iw])
            assert hw == orc.halfwidth(float(zs[iz]), float(ws[iw]))


@pytest.mark.parametrize("args", [
    (0, 20, 2, 60, 20, 2, 1024),        # nbins < 1
    (1000, 20, 3, 60, 20, 2, 1024),     # zmax/dz not an integer
    (1000, 20, 2, 60, 20, 3, 1024),     # numbetween not 1 or 2
    (1000, 20, 2, 60, 20, 0, 1024),
    (1000, 20, 2, 60, 20, 2, 1000),     # seg_len not a supported power of two
    (1000, 200, 2, 6000, 20, 2, 1024),  # overlap larger than the segment
    (1000, -1, 2, 60, 20, 2, 1024),
    (1000, 20, 0, 60, 20, 2, 1024),
])
def test_plan_create_rejects(lib, args):
    h = C.c_void_p()
    rc = lib.jerk_plan_create(C.byref(h), *[int(a) if i in (0, 5, 6) else float(a) for i, a in enumerate(args)])
    assert rc == binding.JERK_EINVAL and not h.value


def test_numbetween_one_halves_points_and_bank(lib):
    """numbetween = 1 keeps the integer-bin phase only."""
    a = binding.Plan(1 << 16, 20, 2, 0, 20, 2, 4096).info
    b = binding.Plan(1 << 16, 20, 2, 0, 20, 1, 4096).info
    assert b.numbetween == 1 and b.points * 2 == a.points and b.flops_per_search * 2 == a.flops_per_search
    assert (b.bank_bytes - 256) * 2 == a.bank_bytes - 256 and (b.step, b.nseg, b.hw_max) == (a.step, a.nseg, a.hw_max)


def test_bank_range_bytes(lib):
    p = binding.Plan(1 << 16, 200, 2, 600, 20, 2, 4096)
    T = p.info.ntemplates
    full = lib.jerk_bank_bytes_range(p._h, T)
    assert full == p.info.bank_bytes
    part = lib.jerk_bank_bytes_range(p._h, T // 8 + 1)
    assert part - (full - T * 2 * 4096 * 8) == (T // 8 + 1) * 2 * 4096 * 8       # tables of the whole grid + this rank's filters
    assert lib.jerk_bank_bytes_range(p._h, T + 1) == 0
    assert lib.jerk_strerror(binding.JERK_EOVERFLOW).startswith(b"JERK_EOVERFLOW")


def test_null_arguments(lib):
    assert lib.jerk_plan_create(None, 10, 1.0, 1.0, 1.0, 1.0, 2, 1024) == binding.JERK_EINVAL
    assert lib.jerk_plan_info(None, None) == binding.JERK_EINVAL
    assert lib.jerk_templates(None, None, 0, None) == binding.JERK_EINVAL
    assert lib.jerk_strerror(binding.JERK_ESTATE).startswith(b"JERK_ESTATE")
    assert lib.jerk_plane_bytes(10, 3, 2) == 10 * 2 * 3 * 2 * 4


def test_search_before_templates_is_estate(lib):
    p = binding.Plan(4096, 20, 2, 60, 20, 2, 1024)
    fake = C.c_void_p(4096)     # never dereferenced: the state check comes first
    rc = lib.jerk_search_candidates(p._h, fake, 20.0, fake, 10, fake, fake, int(p.info.work_bytes), None)
    assert rc == binding.JERK_ESTATE


def test_synth_configs_are_deterministic():
    cfg = synth.config(1)
    a = synth.make_spectrum(cfg)
    b = synth.make_spectrum(synth.config(1))
    assert a.dtype == np.complex64 and a.size == 32768 and np.array_equal(a, b)
    assert cfg.signals == [(5000.25, 10.0, 40.0, 50.0)]
    # block normalisation: unit mean power per 1000-bin block (reading S15)
    blk = a[3000:4000].astype(np.complex128)
    assert abs(np.mean(np.abs(blk) ** 2) - 1.0) < 1e-5


def test_seg_len_zero_is_the_library_choice(lib):
    p = binding.Plan(1 << 20, 200.0, 2.0, 600.0, 20.0, 2, 0)
    assert p.info.seg_len == 4096 and p.info.step == 4096 - 2 * 258
    assert binding.Plan(32768, 20.0, 2.0, 60.0, 20.0, 2, 0).info.seg_len == 1024      # config 1: too few work items for the two-pass kernel
    assert binding.Plan(1 << 20, 100.0, 2.0, 300.0, 20.0, 2, 0).info.seg_len == 4096  # config 2
    with pytest.raises(binding.JerkError):
        binding.Plan(1 << 20, 200.0, 2.0, 600.0, 20.0, 2, 512)


def test_overlap_classes_of_the_plan(lib):
    """Host logic of the overlap classes: the zmax 200 / wmax 600 grid splits into 16 classes whose own
    segmentations add up to fewer (segment, template-phase) units than the nominal ceil(nbins/step) * 2T of SURVEY.md
    8(d) -- recomputed here from the oracle's half-widths -- and small grids keep one class with the nominal count."""
    import math
    nbins = 1 << 22
    p = binding.Plan(nbins, 200, 2, 600, 20, 2, 4096)
    i = p.info
    assert i.nclasses == 16 and i.hw_max == 258 and i.step == 3580
    zs, ws = orc.grid_values(200, 2), orc.grid_values(600, 20)
    hws = sorted(orc.halfwidth(float(z), float(w)) for w in ws for z in zs)
    lo, hi = hws[0], hws[-1]
    width = (hi - lo + 16) // 16
    units = 0
    for k in range(16):
        members = [h for h in hws if (h - lo) // width == k]
        if not members:
            continue
        hw, step = max(members), 4096 - 2 * max(members)
        base = -(i.c_max + hw)
        base -= base & 1
        nseg = -((nbins + i.c_max - hw - base) // -step)
        units += nseg * 2 * len(members)
    assert units == i.units_per_search
    nominal = math.ceil(nbins / i.step) * 2 * i.ntemplates
    assert 0.93 < units / nominal < 0.95
    assert 0.93 < i.flops_per_search_executed / i.flops_per_search < 0.95
    small = binding.Plan(32768, 20, 2, 60, 20, 2, 4096).info
    assert small.nclasses == 1 and small.units_per_search == small.nseg * 2 * small.ntemplates


def test_template_units_balance_the_strong_scaling_split(lib):
    """jerk_template_units (SURVEY.md 8(e), strong scaling): per-template units sum to units_per_search, follow the overlap
    classes (wider templates, more units), and shard.template_range cut at equal units leaves <= 1 % between 8 ranks on
    the config-3 grid where the equal-count split leaves 6 %."""
    from paper_1911_01353_b200 import shard
    cfg = synth.config(3)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, 4096)
    u = plan.template_units()
    T = int(plan.info.ntemplates)
    assert u.shape == (T,) and int(u.sum()) == int(plan.info.units_per_search)
    # recomputed from the oracle's half-widths: a template of a wider class never has fewer units
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    hw = np.array([orc.halfwidth(float(z), float(w)) for w in ws for z in zs])
    order = np.argsort(hw, kind="stable")
    assert np.all(np.diff(u[order]) >= 0)
    for world in (2, 3, 4, 8):
        parts = [shard.template_range(T, world, r, u) for r in range(world)]
        assert parts[0][0] == 0 and parts[-1][0] + parts[-1][1] == T
        assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(world - 1))
        work = [int(u[lo:lo + cnt].sum()) for lo, cnt in parts]
        assert max(work) / min(work) <= 1.01, (world, work)
    flat = [int(u[lo:lo + cnt].sum()) for lo, cnt in (shard.template_range(T, 8, r) for r in range(8))]
    assert max(flat) / min(flat) > 1.04
    # a small grid is one class: equal units per template, the balanced split equals the equal-count split up to a template
    c1 = synth.config(1)
    p1 = binding.Plan(c1.nbins, c1.zmax, c1.dz, c1.wmax, c1.dw, 2, 1024)
    u1 = p1.template_units()
    assert len(set(u1.tolist())) == 1
    for r in range(4):
        a, b = shard.template_range(u1.size, 4, r, u1), shard.template_range(u1.size, 4, r)
        assert abs(a[0] - b[0]) <= 1 and abs(a[1] - b[1]) <= 1
    # more ranks than templates: every template is assigned exactly once, surplus ranks get empty ranges
    uu = np.array([5, 5, 5], dtype=np.int64)
    parts = [shard.template_range(3, 7, r, uu) for r in range(7)]
    seen = np.zeros(3, dtype=int)
    for lo, cnt in parts:
        seen[lo:lo + cnt] += 1
    assert (seen == 1).all()
