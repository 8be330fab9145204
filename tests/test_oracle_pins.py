"""Pins P1-P3 of DESIGN.md: the oracle against hand-computed worked examples
(tests/golden/hand_toys.txt) — values fixed by PAPER.md eq. (2), (4), (6), Alg. 2."""
import os
import numpy as np
import pytest
from oracle import lgo
from helpers import mk_instance

HERE = os.path.dirname(os.path.abspath(__file__))


def golden(tag):
    out = {}
    for l in open(os.path.join(HERE, "golden", "hand_toys.txt")):
        p = l.split()
        if p and p[0] == tag:
            out[p[1]] = [float(x) for x in p[2:]]
    return out


def toy_a(n_tours=1, **kw):
    return mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 60)], [2.0], [10.0, 10.0], n_tours, **kw)


PLAN_A = dict(bp_tour=[0], bp_pos=[0], field_bp=[0, 0], field_pos=[0, 1], hu_tour=[0], su_tour=[0, 0])


def test_toy_a_values():
    g = golden("A")
    o = lgo.Oracle(toy_a())
    r = o.score(PLAN_A)
    assert r["feasible"]
    assert r["route"][0] == g["route_km"][0]
    assert list(r["shuttles"]) == g["shuttles"]
    assert r["L_HU"] == g["L_HU"][0] and r["L_eSU"] == g["L_eSU"][0] and r["L_lSU"] == g["L_lSU"][0]
    assert r["path"] == g["path_km"][0]
    assert r["makespan"] == g["makespan_h"][0]
    assert r["cost"] == g["cost"][0]
    assert r["E"][0] == pytest.approx(g["E_h"][0], rel=1e-14)
    assert r["wait"][0] == pytest.approx(g["wait_h"][0], rel=1e-13)


def test_toy_a_reversed_order_and_infeasible():
    # Visiting B first: HQ->B (10) ->A (5) ->HQ (5): same length; shuttles follow the field.
    o = lgo.Oracle(toy_a())
    r = o.score(dict(PLAN_A, field_pos=[1, 0]))
    assert r["route"][0] == 20 and r["path"] == 154 and list(r["shuttles"]) == [3, 4]
    # demand 66 t > 65 t supplied => discarded: +inf, flag 0
    o2 = lgo.Oracle(mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 66)], [2.0], [10.0, 10.0], 1))
    r2 = o2.score(PLAN_A)
    assert not r2["feasible"] and np.isinf(r2["cost"]) and np.isinf(r2["path"]) and np.isinf(r2["makespan"])
    # demand exactly 65 t is met: eq. (2) is ">="
    o3 = lgo.Oracle(mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 65)], [2.0], [10.0, 10.0], 1))
    assert o3.score(PLAN_A)["feasible"]


def test_toy_a_weights_and_velocities():
    # cost = w_path*path + w_time*makespan
    r = lgo.Oracle(toy_a(w_path=2.0, w_time=10.0)).score(PLAN_A)
    assert r["cost"] == 2 * 154 + 10 * 2.0
    # v_HU enters the completion time only; v_SU enters E (t_edge) only
    r = lgo.Oracle(toy_a(v_hu_road_kmh=20.0)).score(PLAN_A)
    assert r["makespan"] == 20 / 20 + 1.5 and r["E"][0] == pytest.approx(0.325, rel=1e-14)
    r = lgo.Oracle(toy_a(v_su_road_kmh=20.0)).score(PLAN_A)
    assert r["makespan"] == 2.0 and r["E"][0] == pytest.approx(0.65, rel=1e-14)
    # one more SU: L_eSU grows by the route, shuttle counts use ceil(s*n/C) with C = 30
    r = lgo.Oracle(mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 60)], [2.0],
                               [10.0, 10.0, 10.0], 1)).score(dict(PLAN_A, su_tour=[0, 0, 0]))
    assert list(r["shuttles"]) == [3, 4] and r["L_eSU"] == 3 * 20 + 47
    # a second HU on the tour adds its rate and its route length
    r = lgo.Oracle(mk_instance((0, 0), [(3, 4, 25, 1), (6, 8, 40, 2)], [(6, 0, 60)], [2.0, 1.0],
                               [10.0, 10.0], 1)).score(dict(PLAN_A, hu_tour=[0, 0]))
    assert r["L_HU"] == 40 and r["makespan"] == 0.5 + 3 / 3.0
    assert r["wait"][0] == pytest.approx(0.325 - 0.008 * 10 / 2, rel=1e-13)


def toy_d():
    fields = [(3, 4, 25, 1), (6, 8, 40, 2), (0, -5, 30, 3), (12, -5, 20, 1), (12, -16, 50, 4)]
    bps = [(6, 0, 60), (0, -10, 50), (12, -10, 50)]
    inst = mk_instance((0, 0), fields, bps, [2.0, 1.0, 3.0], [10, 10, 20, 20, 10], 2, su_fill_h_per_t=0.01)
    plan = dict(bp_tour=[0, 1, 1], bp_pos=[0, 0, 1], field_bp=[0, 0, 1, 1, 2], field_pos=[0, 1, 0, 1, 0],
                hu_tour=[0, 1, 1], su_tour=[0, 0, 1, 1, 1])
    return inst, plan


def test_toy_d_values():
    g = golden("D")
    inst, plan = toy_d()
    r = lgo.Oracle(inst).score(plan)
    assert r["feasible"]
    assert list(r["route"]) == g["route_km"]
    assert list(r["shuttles"]) == g["shuttles"]
    assert list(r["L"]) == g["L_tour_total"]
    assert r["path"] == g["path_km"][0]
    assert list(r["T"]) == pytest.approx(g["T_h"], rel=1e-15)
    assert r["makespan"] == pytest.approx(g["makespan_h"][0], rel=1e-15)
    assert r["cost"] == pytest.approx(g["cost"][0], rel=1e-15)
    assert r["E"] == pytest.approx(g["E_h"], rel=1e-14)
    assert (r["L_HU"], r["L_eSU"], r["L_lSU"]) == (g["L_HU"][0], g["L_eSU"][0], g["L_lSU"][0])
    assert list(r["su_tour_final"]) == plan["su_tour"] and r["moves"] == 0
    assert list(r["bp_supply_q"]) == [65 * 1024, 50 * 1024, 50 * 1024]
    # swapping the BP order on tour 1 changes the route: HQ->F4 (20)->F2 (sqrt(144+121))...
    r2 = lgo.Oracle(inst).score(dict(plan, bp_pos=[0, 1, 0]))
    assert r2["route"][1] == pytest.approx(20 + np.sqrt(12**2 + 11**2) + 12 + 13, rel=1e-15)
    # one quantum short on BP2 => infeasible
    inst.bp_demand_t[2] = 50 + 1 / 1024
    assert not lgo.Oracle(inst).score(plan)["feasible"]


def test_trace_b_alg2_two_tours():
    # P2: kappa=0.01, 1 HU per tour, E=(0.5,0.1), U_0={10}, U_1={10,20,30}
    cap = np.array([10, 10, 20, 30]) * 1024
    moves, su, W = lgo.su_local_min([0.5, 0.1], [1, 1], cap, [0, 1, 1, 1], 0.01)
    assert moves == 2
    assert list(su) == [0, 1, 0, 0]          # tour 0 = {10,20,30}, tour 1 keeps the second 10
    assert W == pytest.approx([0.2, 0.1], abs=1e-12)


def test_trace_c_alg2_three_tours_early_accept():
    # P3: E=(0.5,0.45,0.1), U=({10},{10},{10,20,30}); accepts the smallest unit that
    # pushes T_wait(g_max) below T_wait(g_2nd)
    cap = np.array([10, 10, 10, 20, 30]) * 1024
    moves, su, W = lgo.su_local_min([0.5, 0.45, 0.1], [1, 1, 1], cap, [0, 1, 2, 2, 2], 0.01)
    assert moves == 2
    assert list(su) == [0, 1, 0, 1, 2]
    assert W == pytest.approx([0.4, 0.35, 0.1], abs=1e-12)


def test_alg2_degenerate_cases():
    cap = np.array([10, 20]) * 1024
    # N_T = 1: no-op (R12)
    moves, su, W = lgo.su_local_min([0.3], [1], cap, [0, 0], 0.01)
    assert moves == 0 and W[0] == pytest.approx(0.3 - 0.1)
    # donor has a single SU: it keeps it (R15)
    moves, su, W = lgo.su_local_min([0.9, 0.1], [1, 1], cap, [0, 1], 0.01)
    assert moves == 0 and list(su) == [0, 1]
    # a move that does not lower the maximum is undone (R14): W=(0.5,0.2); moving a 30
    # gives (0.4,0.5): the maximum stays 0.5, not strictly lower => undo, stop.
    cap = np.array([10, 30, 30]) * 1024
    moves, su, W = lgo.su_local_min([0.5, 0.5], [1, 1], cap, [0, 1, 1], 0.01)
    assert moves == 0 and list(su) == [0, 1, 1] and W == pytest.approx([0.5, 0.2], abs=1e-12)
    # ... while E=(0.5,0.49) lets the same move stand: (0.4,0.49), maximum 0.5 -> 0.49
    moves, su, W = lgo.su_local_min([0.5, 0.49], [1, 1], cap, [0, 1, 1], 0.01)
    assert moves == 1 and list(su) == [0, 1, 0] and W == pytest.approx([0.4, 0.49], abs=1e-12)
    # HU count divides the fill-time term (eq. (6), R7)
    # by hand: W = (0.5 - 0.01*(40-30)/4, 0 - 0.01*(20-10)/1) = (0.475, -0.1); neither 10 t unit of tour 1 brings
    # tour 0 below -0.1 (0.5 - 0.01*20/4 = 0.45), so the largest by (capacity, unit) = unit 3 moves: (0.45, 0.0),
    # maximum 0.475 -> 0.45, kept; then the donor is down to one SU.  With n_HU = 1 the waits would be 0.4 -> 0.3.
    moves, su, W = lgo.su_local_min([0.5, 0.0], [4, 1], np.array([10, 30, 10, 10]) * 1024, [0, 0, 1, 1], 0.01)
    assert moves == 1 and list(su) == [0, 0, 1, 0] and W == pytest.approx([0.45, 0.0], abs=1e-12)
    W0 = lgo.su_local_min([0.5], [4], np.array([10, 30]) * 1024, [0, 0], 0.01)[2][0]
    assert W0 == pytest.approx(0.5 - 0.01 * 10 / 4)


def test_distance_and_quantisation():
    o = lgo.Oracle(mk_instance((0, 0), [(3, 4, 0.5 / 1024, 1.5 / 1024), (1e3, 1e-3, 2.5 / 1024, 1)],
                               [(6, 0, 0)], [2.0], [10.0], 1))
    assert o.distance(0, 2) == 5.0 and o.distance(2, 0) == 5.0 and o.distance(2, 2) == 0.0
    assert o.distance(0, 1) == 6.0 and o.distance(1, 2) == 5.0     # vertex order HQ, BPs, fields
    d = o.distance(0, 3)
    assert d == np.sqrt(1e3 * 1e3 + 1e-3 * 1e-3)
    # round-half-even on Q = 1024 (R18)
    assert list(o.quanta(0)) == [0, 2] and list(o.quanta(1)) == [2, 1024]
    assert list(o.quanta(3)) == [2048] and list(o.quanta(4)) == [10240]


def test_create_rejects_bad_input():
    ok = toy_a()
    for bad in (dict(n_tours=2), dict(n_tours=0), dict(v_hu_road_kmh=0.0), dict(v_su_road_kmh=float("nan")),
                dict(su_fill_h_per_t=-1.0)):
        with pytest.raises(lgo.OracleError):
            lgo.Oracle(toy_a(**bad))
    inst = toy_a(); inst.su_capacity_t[0] = 0.0
    with pytest.raises(lgo.OracleError):
        lgo.Oracle(inst)
    inst = toy_a(); inst.field_supply_t[0] = -1.0
    with pytest.raises(lgo.OracleError):
        lgo.Oracle(inst)
    inst = toy_a(); inst.field_supply_t[0] = 3e6     # s_q*N_SU + sum c_q >= 2^32
    with pytest.raises(lgo.OracleError) as e:
        lgo.Oracle(inst)
    assert e.value.code == -2
    lgo.Oracle(ok)


# ---- P9: the decoder's draw ORDER, derived by hand from published random words (S1-S3; PAPER.md:L233,
#      "identical random process control"; L116-118 the decision variables the draws fix).  The invariants and the
#      chi-square tests of test_oracle_invariants.py would still pass with a wrong draw index that keeps the
#      distribution; these values would not.

def _kat_row0():
    for l in open(os.path.join(HERE, "golden", "philox4x32_10_kat.txt")):
        p = l.split()
        if p and not l.startswith("#"):
            return [int(x, 16) for x in p]
    raise AssertionError("no known-answer vector")


def test_bp_partition_of_seed0_id0_from_the_published_vector():
    """Stream 0 / block 0 of (seed 0, id 0) has counter (0, 0, 0, 0) and key (0, 0): exactly the first published
    known-answer vector of Philox4x32-10, output words w = (6627e8d5, e169c58d, bc57ac4c, 9b00dbd8).
    S2 with n = N_B = 3 items, k = N_T = 2 bins, below(x, m) = floor(x m / 2^32):
      a = [0 1 2]
      i = 2: j = below(w0, 3) = floor(0x6627e8d5 * 3 / 2^32) = floor(1.197) = 1 -> swap a[2], a[1] -> a = [0 2 1]
      i = 1: j = below(w1, 2) = top bit of 0xe169c58d            = 1 -> swap a[1], a[1] -> a = [0 2 1]
      consumption p = 0 reads a[2] = BP 1 -> bin 0 = tour 0, position 0
                  p = 1 reads a[1] = BP 2 -> bin 1 = tour 1, position 0
                  p = 2 reads a[0] = BP 0 -> bin below(draw 2 + (2 - 2) = w2, 2) = top bit of 0xbc57ac4c = 1 -> tour 1, position 1
    so bp_tour = [1 0 1] and bp_pos = [1 0 0] (indexed by BP)."""
    kat = _kat_row0()
    assert kat[:6] == [0, 0, 0, 0, 0, 0] and kat[6:] == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    w = kat[6:]
    assert [(w[0] * 3) >> 32, (w[1] * 2) >> 32, (w[2] * 2) >> 32] == [1, 1, 1]
    from paper_1909_10286_b200 import workloads as wl
    inst = wl.make("toy")
    assert (inst.n_bps, inst.n_tours, inst.n_fields) == (3, 2, 11)
    plan = lgo.Oracle(inst).decode_batch(0, first_id=0, n=1)
    assert plan["bp_tour"][0].tolist() == [1, 0, 1]
    assert plan["bp_pos"][0].tolist() == [1, 0, 0]


def test_first_field_swaps_of_seed0_id0_from_the_curand_header(tmp_path):
    """Stream 3 (field permutation) and stream 4 (extras), block 0 of (seed 0, id 0): counters (0, 0, 3, 0) and
    (0, 0, 4, 0), key (0, 0).  The words come from NVIDIA's cuRAND header compiled for the host (an implementation that
    is neither the oracle's nor the kernels').
    S3 over N_F = 11 fields: i = 10: j = below(w0, 11), swap a[10], a[j]; i = 9: j = below(w1, 10), swap a[9], a[j].
    a[10] and a[9] are final after their steps and are the first two fields consumed.  The first BP in plan order is
    BP 1 (tour 0's only BP, see the pin above), the second BP 2 (first on tour 1).  Field a[10] goes to BP 1 at
    position 0.  In the toy instance any one field covers BP 1's demand many times over, so the minimal prefix ends
    there and the first extras draw x = word 0 of stream 4 decides where a[9] goes: x < extra_field_thresh -> BP 1,
    position 1; otherwise BP 1 is closed and a[9] opens BP 2 at position 0."""
    import shutil, subprocess, textwrap
    if shutil.which("nvcc") is None:
        pytest.skip("nvcc not found")
    src = tmp_path / "w.cu"
    src.write_text(textwrap.dedent(r"""
        #include <cstdio>
        #include <cuda_runtime.h>
        #define QUALIFIERS static inline __host__ __device__
        #include <curand_philox4x32_x.h>
        int main() {
          for (unsigned s = 3; s <= 4; ++s) {
            uint4 r = curand_Philox4x32_10(make_uint4(0u, 0u, s, 0u), make_uint2(0u, 0u));
            printf("%08x %08x %08x %08x\n", r.x, r.y, r.z, r.w);
          }
          return 0;
        }"""))
    exe = tmp_path / "w"
    r = subprocess.run(["nvcc", "-O1", "-o", str(exe), str(src)], capture_output=True, text=True)
    if r.returncode != 0:
        pytest.skip("cuRAND header does not compile for the host here: " + r.stderr[-300:])
    words = [int(x, 16) for x in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    w3, w4 = words[:4], words[4:]
    a = list(range(11))
    j = (w3[0] * 11) >> 32; a[10], a[j] = a[j], a[10]
    j = (w3[1] * 10) >> 32; a[9], a[j] = a[j], a[9]
    from paper_1909_10286_b200 import workloads as wl
    inst = wl.make("toy")
    assert inst.field_supply_t.min() > 2.0 * inst.bp_demand_t[1]          # one field is a complete minimal prefix of BP 1
    second = (1, 1) if w4[0] < inst.extra_field_thresh else (2, 0)
    plan = lgo.Oracle(inst).decode_batch(0, first_id=0, n=1)
    fb, fp = plan["field_bp"][0], plan["field_pos"][0]
    assert (int(fb[a[10]]), int(fp[a[10]])) == (1, 0)
    assert (int(fb[a[9]]), int(fp[a[9]])) == second
