"""Seeded synthetic instance generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the oracle (tests, bench.py) and therefore
holds none of the method's arithmetic: it only draws coordinates, areas, yields,
demands, rates and capacities with the shapes and distributions the configs state
(§3.1 for the paper's own recipe: uniform locations in a square, HQ at
the origin, straight-line edges; Table 1 PAPER.md:L51-65 for the unit parameters).
The paper's 10 random location sets are unpublished; these inputs stand in for them
(recipe restated in DESIGN.md §"Input recipe").

Draw order per config (numpy default_rng(1909102860 + k), k = config index):
BPs (x then y), field cluster centres if any, fields (x, y), areas, yields,
Dirichlet shares, HU rates, SU capacities.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
import numpy as np

SEED_BASE = 1909102860


@dataclass
class Instance:
    """Plain host-side description of one problem instance."""
    name: str
    hq: tuple            # (x, y) km; "HQ ... at the origin"
    field_xy: np.ndarray  # [N_F, 2] km
    field_supply_t: np.ndarray  # s_f (t)      eq. (2)/(3) PAPER.md:L79-85
    field_area_ha: np.ndarray   # h_f (ha)
    bp_xy: np.ndarray     # [N_B, 2] km
    bp_demand_t: np.ndarray     # d_b^min (t)  eq. (2)
    hu_rate_ha_per_h: np.ndarray  # per unit   PAPER.md:L96 (ii)
    su_capacity_t: np.ndarray     # per unit
    n_tours: int
    v_hu_road_kmh: float = 40.0   # Table 1
    v_su_road_kmh: float = 40.0   # Table 1
    v_infield_kmh: float = 15.0   # configs only; stored, unused (R24)
    su_fill_h_per_t: float = 0.008  # Table 1: 6 min/12.5 t, 8 min/16.5 t (R8)
    w_path: float = 1.0
    w_time: float = 1.0
    extra_field_thresh: int = 0x40000000
    flags: int = 0
    budget: int = 0       # number of candidates the config asks for
    seed: int = 0         # candidate seed

    @property
    def n_fields(self): return int(self.field_xy.shape[0])
    @property
    def n_bps(self): return int(self.bp_xy.shape[0])
    @property
    def n_hu(self): return int(self.hu_rate_ha_per_h.shape[0])
    @property
    def n_su(self): return int(self.su_capacity_t.shape[0])


_CONFIGS = {
    #  name      k  side  N_F  N_B  N_T N_HU N_SU dem   hu_rate     su_cap     homog  clusters budget
    "toy":    (0,  40.0,  11,   3,  2,   4,   8, 0.90, (1.5, 3.0), (15., 30.), True,  0, 1 << 16),
    "small":  (1,  80.0,  40,   5,  3,   8,  20, 0.90, (1.5, 3.0), (15., 30.), False, 0, 1 << 24),
    "medium": (2, 100.0, 100,   8,  5,  12,  36, 0.95, (1.5, 3.0), (15., 30.), False, 4, 1 << 28),
    "large":  (3, 150.0, 250,  12,  8,  20,  60, 0.90, (1.0, 4.0), (10., 40.), False, 0, 1 << 30),
    "sweep":  (4, 200.0, 500,  20, 10,  30, 100, 0.90, (1.0, 4.0), (10., 40.), False, 0, 1 << 32),
}
CONFIG_NAMES = tuple(_CONFIGS)


def make(name: str) -> Instance:
    """Build one of the five configs (or 'toy_brute', the N_B=2, N_F=6 sub-instance)."""
    if name == "toy_brute":
        return _toy_brute()
    if name == "paper_scale":
        return _paper_scale()
    k, side, nf, nb, nt, nhu, nsu, dem, hr, sc, homog, ncl, budget = _CONFIGS[name]
    rng = np.random.default_rng(SEED_BASE + k)
    bp_xy = np.stack([rng.uniform(0, side, nb), rng.uniform(0, side, nb)], axis=1)
    if ncl:
        centres = rng.uniform(20.0, 80.0, (ncl, 2))
        which = rng.integers(0, ncl, nf)
        fx = np.clip(centres[which, 0] + 10.0 * rng.standard_normal(nf), 0.0, side)
        fy = np.clip(centres[which, 1] + 10.0 * rng.standard_normal(nf), 0.0, side)
        field_xy = np.stack([fx, fy], axis=1)
    else:
        field_xy = np.stack([rng.uniform(0, side, nf), rng.uniform(0, side, nf)], axis=1)
    area = rng.uniform(5.0, 40.0, nf)
    yield_t_ha = rng.uniform(30.0, 50.0, nf)
    supply = area * yield_t_ha
    shares = rng.dirichlet(np.ones(nb))
    demand = dem * supply.sum() * shares
    if homog:
        hu = np.full(nhu, rng.uniform(*hr))
        su = np.full(nsu, rng.uniform(*sc))
    else:
        hu = rng.uniform(hr[0], hr[1], nhu)
        su = rng.uniform(sc[0], sc[1], nsu)
    return Instance(name=name, hq=(0.0, 0.0), field_xy=field_xy, field_supply_t=supply,
                    field_area_ha=area, bp_xy=bp_xy, bp_demand_t=demand,
                    hu_rate_ha_per_h=hu, su_capacity_t=su, n_tours=nt, budget=budget)


def _toy_brute() -> Instance:
    """First 2 BPs / 6 fields of Toy; demands rescaled to 0.9 x the 6 fields' supply."""
    t = make("toy")
    supply = t.field_supply_t[:6].copy()
    d = t.bp_demand_t[:2].copy()
    d = d / d.sum() * 0.9 * supply.sum()
    return replace(t, name="toy_brute", field_xy=t.field_xy[:6].copy(), field_supply_t=supply,
                   field_area_ha=t.field_area_ha[:6].copy(), bp_xy=t.bp_xy[:2].copy(),
                   bp_demand_t=d, budget=1 << 24)


def _paper_scale() -> Instance:
    """Shape of the paper's own workload (Table 1): 1200 fields,
    20 BPs, 7 tours, 7 HUs at 2.5 ha/h, 14 SUs of 12.5 t + 28 of 16.5 t, 80x80 km,
    h_f = 3 + 4u ha.  The paper measures supply and demand in ha (s_f = h_f, d_b = 250 ha);
    here both are converted to tonnes with eq. (3)'s c_conv = 40 t/ha so that eq. (4)'s
    shuttle counts use the capacities of Table 1 (t)."""
    rng = np.random.default_rng(SEED_BASE + 5)
    nf, nb, side = 1200, 20, 80.0
    bp_xy = np.stack([rng.uniform(0, side, nb), rng.uniform(0, side, nb)], axis=1)
    field_xy = np.stack([rng.uniform(0, side, nf), rng.uniform(0, side, nf)], axis=1)
    area = 3.0 + 4.0 * rng.uniform(0, 1, nf)
    supply = 40.0 * area                      # eq. (3), c_conv = 40 t/ha
    demand = np.full(nb, 250.0 * 40.0)        # 250 ha of corn per BP, in t
    hu = np.full(7, 2.5)
    su = np.concatenate([np.full(14, 12.5), np.full(28, 16.5)])
    return Instance(name="paper_scale", hq=(0.0, 0.0), field_xy=field_xy, field_supply_t=supply,
                    field_area_ha=area, bp_xy=bp_xy, bp_demand_t=demand, hu_rate_ha_per_h=hu,
                    su_capacity_t=su, n_tours=7, budget=1 << 24)


def sample_ids(budget: int, n: int, seed: int = 12345) -> np.ndarray:
    """n ids spread over [0, budget): uniform draws (so ids >= 2^31 / 2^32-ish appear for
    the big configs).  Plain numpy; no method arithmetic."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, budget, n, dtype=np.uint64)
