"""Host-side pieces of SURVEY 8(f) that need no GPU: the perf_analyzer normalisation (NEXT-3) and the autoscaler policy
(NEXT-2), each pinned to what the paper prints."""
import numpy as np

from paper_2312_06838_b200 import autoscale as A
from paper_2312_06838_b200 import perf


def test_normalisation_example_of_the_paper():
    """'a BDT with 25 FP32 inputs, batch size of 500, and a total network latency of 14,800 us, would have a
    normalized value of 1.184 us'."""
    assert abs(perf.normalised_us(14800.0, 25, 500) - 1.184) < 1e-12
    assert perf.normalised_us(800.0, 8 * 100, 1) == 1.0                  # Table C2: ParticleNet input shape 8 x 100


def test_request_pool_cuts_whole_requests():
    import synth
    b = synth.make_particlenet_batch(n_jets=100)
    rfj = perf.request_pool(b, 16)
    assert rfj.tolist() == [0, 16, 32, 48, 64, 80, 96] and rfj.dtype == np.int32


def scale_times(samples, p=A.SP2):
    sc = A.Autoscaler(p=p)
    ev, n = [], sc.instances
    for q in samples:
        m = sc.step(q)
        if m != n:
            ev.append((sc.t, m - n))
            n = m
    return ev


def test_scale_up_rule_of_sp2():
    """L105: above 400 ms for four consecutive 15 s samples and >= 3 minutes since the last scale-up: one more server.  With
    the queue time above the threshold from the start: t = 60 s (4th sample), then every 180 s (Table A1 periodSeconds)."""
    ev = scale_times([900.0] * 40)
    assert ev[:3] == [(60.0, 1), (240.0, 1), (420.0, 1)]
    assert all(d == 1 for _, d in ev)                                   # policies.value 1: one server at a time
    # analysis points are 30 s averages: samples 900 900 100 100 900 900 900 give points 900 900 500 100 500 900 900, i.e. runs
    # of 3 and 3 consecutive points above 400 ms: no scale-up; one more high sample completes a run of four at t = 120 s
    assert scale_times([900, 900, 100, 100, 900, 900, 900]) == []
    assert scale_times([900, 900, 100, 100, 900, 900, 900, 900]) == [(120.0, 1)]


def test_window_is_two_samples():
    """App. A: 30 s data collection window = 2 consecutive 15 s measurements."""
    sc = A.Autoscaler()
    sc.step(0.0); sc.step(900.0)
    assert sc.windowed() == 450.0
    sc.step(300.0)
    assert sc.windowed() == 600.0


def test_scale_down_rule_and_limits():
    """L105: below 400 ms for 40 consecutive samples and >= 1 minute since the last scale-down: one server less; never below
    one; at most 10 (App. A: ten MIG instances)."""
    sc = A.Autoscaler(instances=3)
    t_down = []
    for i in range(60):
        n0 = sc.instances
        if sc.step(10.0) < n0:
            t_down.append(sc.t)
    assert t_down == [600.0, 660.0] and sc.instances == 1               # 40th sample, then scaleDown periodSeconds = 60
    ev = scale_times([5000.0] * 200)
    assert len(ev) == 9 and ev[-1][0] == 60.0 + 8 * 180.0               # 1 -> 10 instances, then the cap holds


def test_no_flapping_around_the_threshold():
    """App. A: the long scale-down window exists to avoid 'flapping' while the queue time oscillates around the threshold."""
    osc = [600.0, 600.0, 100.0, 100.0] * 30
    assert all(d > 0 for _, d in scale_times(osc)) or scale_times(osc) == []


def test_sp1_is_more_eager_than_sp2():
    """L105: SP1 used a 100 ms threshold; a 250 ms queue time scales SP1 up and leaves SP2 alone."""
    assert scale_times([250.0] * 20, A.SP1)[0] == (60.0, 1)
    assert scale_times([250.0] * 20, A.SP2) == []


def test_simulated_ramp_scales_up_then_down():
    """The shape of Figs. 7-9: instances follow a client ramp one at a time, throughput grows with serving instances, and the
    service returns to one instance after the load stops."""
    tr = A.simulate(lambda t: min(120.0, t / 5.0) if t < 2500 else 0.0, service_rate_per_instance=5.0,
                    request_rate_per_worker=1.0, duration_s=4500.0)
    inst = [r["instances"] for r in tr]
    assert max(inst) == 10 and inst[-1] == 1
    assert all(abs(a - b) <= 1 for a, b in zip(inst, inst[1:]))
    peak = max(r["throughput"] for r in tr)
    assert 45.0 <= peak <= 50.0 + 1e-9                                  # 10 instances x 5 requests/s (App. A: ~5 per instance)
    ups = [r["t"] for a, r in zip(tr, tr[1:]) if r["instances"] > a["instances"]]
    assert all(b - a >= 180.0 for a, b in zip(ups, ups[1:]))
