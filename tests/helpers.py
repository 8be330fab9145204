"""Small helpers shared by tests (no method arithmetic)."""
from types import SimpleNamespace
import numpy as np


def mk_instance(hq, fields, bps, hu, su, n_tours, **kw):
    """fields: [(x,y,supply_t,area_ha)], bps: [(x,y,demand_t)]."""
    f = np.asarray(fields, dtype=np.float64).reshape(-1, 4)
    b = np.asarray(bps, dtype=np.float64).reshape(-1, 3)
    d = dict(name="hand", hq=tuple(hq), field_xy=f[:, :2].copy(), field_supply_t=f[:, 2].copy(),
             field_area_ha=f[:, 3].copy(), bp_xy=b[:, :2].copy(), bp_demand_t=b[:, 2].copy(),
             hu_rate_ha_per_h=np.asarray(hu, dtype=np.float64), su_capacity_t=np.asarray(su, dtype=np.float64),
             n_tours=n_tours, v_hu_road_kmh=40.0, v_su_road_kmh=40.0, v_infield_kmh=15.0,
             su_fill_h_per_t=0.008, w_path=1.0, w_time=1.0, extra_field_thresh=0x40000000, flags=0)
    d.update(kw)
    ns = SimpleNamespace(**d)
    ns.n_fields, ns.n_bps = f.shape[0], b.shape[0]
    ns.n_hu, ns.n_su = len(ns.hu_rate_ha_per_h), len(ns.su_capacity_t)
    return ns
