"""Teacher/student problem set-up computed with the ORACLE (test infrastructure only).

Given a `Workload` (structures + model) this produces what a parity run needs, following the
input recipe of DESIGN.md:  teacher theta -> labels E, F, W (oracle fp64 forward with the
teacher's own scaler);  student theta (rounded to fp32 once; both sides use those values) and
the student's scaler (Eq. 2) that is injected into the CUDA library with nep_set_scaler.
No value here ever comes from the CUDA path.
"""
from __future__ import annotations

import dataclasses

import numpy as np

from . import nep_oracle as O


@dataclasses.dataclass
class Problem:
    workload: object
    data: O.OracleData          # neighbour lists + labels attached
    theta_teacher: np.ndarray   # float64
    scaler_teacher: np.ndarray
    theta: np.ndarray           # student, float64 holding fp32-representable values
    scaler: np.ndarray          # student scaler, float64
    E: np.ndarray
    F: np.ndarray
    W: np.ndarray


def _draw(workload, data, seed):
    from paper_2606_19557_b200.workloads import ParamDraw
    pd = ParamDraw(workload.model, seed)
    th = pd.coefficients()
    q = O.descriptors(data, th)
    s = O.scaler(q)
    th = pd.network((q * s).mean(axis=0))
    return th.copy(), s


def make_problem(workload) -> Problem:
    data = O.OracleData(workload.model, workload.structures)
    th_t, s_t = _draw(workload, data, workload.seeds["teacher"])
    E, F, W = O.forward(data, th_t, s_t)
    th_s, s_s = _draw(workload, data, workload.seeds["student"])
    th_s = th_s.astype(np.float32).astype(np.float64)
    data.set_labels(E, F, W)
    return Problem(workload, data, th_t, s_t, th_s, s_s, E, F, W)
