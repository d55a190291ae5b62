"""ORACLE — test infrastructure only.

Plain CPU McMurchie–Davidson implementation of what the hot path computes (Appendix A,
eqs. 12–19).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports nothing from the
product package and shares no code with the CUDA path.
"""
from .lxo import (  # noqa: F401
    build, boys, boys_ld, eri3_batch, schwarz_aux, schwarz_pair, df_gamma_J, max_threads, ncart, components,
    metric_2c, fit_solve,
)
