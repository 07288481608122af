"""Autoscaler policy simulator (section 3.3.1; L209-L258 App. A, Table A1): the server's metric pipeline and the
Horizontal-Pod-Autoscaler rule that adds or removes inference instances, replayed on a synthetic client ramp.  Host code:
nothing here touches the GPU; the per-instance service rate it needs is a number (measured by bench.py, or given).

Metric pipeline (App. A "Metric collection and analysis parameters"): the queue time per inference request is sampled every
15 s (collection interval = analysis time step); an analysis point is the average over a 30 s window, i.e. over two
consecutive samples (sliding window).
Scaling rule (L105, Table A1), "Scaling Parameters 2": if the windowed queue time exceeds the threshold (400 ms) for four
consecutive analysis points (scaleUp.stabilizationWindowSeconds = 60) and the last scale-up is at least 180 s old
(scaleUp.policies.periodSeconds), one instance is added (policies.type Pods, value 1); if it is below the threshold for 40
consecutive points (scaleDown.stabilizationWindowSeconds = 600) and the last scale-down is at least 60 s old, one is
removed.  "Scaling Parameters 1" is the pre-optimisation setting: a 100 ms threshold (L105); the paper does not print its
windows, so SP1 here differs from SP2 in the threshold only (DESIGN.md readings).
"""
from dataclasses import dataclass, field
from typing import List


@dataclass
class ScalingParameters:
    threshold_ms: float = 400.0
    sample_s: float = 15.0            # metric collection interval = analysis time step
    window_s: float = 30.0            # data collection window (two consecutive samples)
    up_stabilization_s: float = 60.0  # four consecutive points
    up_period_s: float = 180.0
    down_stabilization_s: float = 600.0   # forty consecutive points
    down_period_s: float = 60.0
    min_instances: int = 1
    max_instances: int = 10           # App. A: "the relatively small amount of MIG instances available (10)"


SP2 = ScalingParameters()
SP1 = ScalingParameters(threshold_ms=100.0)


@dataclass
class Autoscaler:
    """Feed one raw queue-time sample (ms) per `sample_s`; step() returns the instance count after the decision."""
    p: ScalingParameters = field(default_factory=ScalingParameters)
    instances: int = 1
    t: float = 0.0
    samples: List[float] = field(default_factory=list)
    above: int = 0
    below: int = 0
    last_up: float = -1e18
    last_down: float = -1e18

    def windowed(self) -> float:
        n = max(1, int(round(self.p.window_s / self.p.sample_s)))
        w = self.samples[-n:]
        return sum(w) / len(w)

    def step(self, queue_ms: float) -> int:
        self.t += self.p.sample_s
        self.samples.append(float(queue_ms))
        q = self.windowed()
        if q > self.p.threshold_ms:
            self.above += 1
            self.below = 0
        else:
            self.below += 1
            self.above = 0
        n_up = int(round(self.p.up_stabilization_s / self.p.sample_s))
        n_down = int(round(self.p.down_stabilization_s / self.p.sample_s))
        if self.above >= n_up and self.t - self.last_up >= self.p.up_period_s and self.instances < self.p.max_instances:
            self.instances += 1
            self.last_up = self.t
        elif self.below >= n_down and self.t - self.last_down >= self.p.down_period_s and self.instances > self.p.min_instances:
            self.instances -= 1
            self.last_down = self.t
        return self.instances


def simulate(workers_at, service_rate_per_instance: float, request_rate_per_worker: float, duration_s: float,
             p: ScalingParameters = SP2, startup_s: float = 30.0, dt: float = 1.0):
    """Fluid model of the service under a client ramp (the shape of Figs. 3, 7-9): workers_at(t) synchronous clients, each
    able to send request_rate_per_worker requests/s when it does not wait; a serving instance handles
    service_rate_per_instance requests/s; a new instance serves only `startup_s` after it is deployed (Fig. A1: the queue
    time is noisy while an instance starts).  Clients are closed-loop, so the backlog is bounded by the number of workers
    (each has one request in flight); queue time of a request = backlog / capacity.  Returns one record per metric sample:
    time, workers, deployed and serving instances, throughput (requests/s) and the windowed queue time (ms)."""
    sc = Autoscaler(p=p)
    trace = []
    backlog = 0.0
    starting = []                     # deployment times of instances that do not serve yet
    t = 0.0
    acc_q, acc_thr, acc_n = 0.0, 0.0, 0
    next_sample = p.sample_s
    while t < duration_s:
        w = float(workers_at(t))
        starting = [x for x in starting if t - x < startup_s]
        serving = max(1, sc.instances - len(starting))
        cap = serving * service_rate_per_instance
        idle = max(0.0, w - backlog)                               # workers that are not waiting for an answer
        offered = min(idle * request_rate_per_worker, idle / dt + cap)
        served = min(cap, backlog / dt + offered)
        backlog = min(w, max(0.0, backlog + (offered - served) * dt))
        acc_q += 1e3 * backlog / cap
        acc_thr += served
        acc_n += 1
        t += dt
        if t + 1e-9 >= next_sample:
            before = sc.instances
            n = sc.step(acc_q / acc_n)
            if n > before:
                starting.append(t)
            elif n < before and starting:
                starting.pop()
            trace.append({"t": t, "workers": w, "instances": n, "serving": serving, "throughput": acc_thr / acc_n,
                          "queue_ms": sc.windowed()})
            acc_q, acc_thr, acc_n = 0.0, 0.0, 0
            next_sample += p.sample_s
    return trace
