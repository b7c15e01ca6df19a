"""Seeded synthetic inputs shared by the oracle and the CUDA path.

This package holds input construction only (tree topologies, rest orientations,
apple placements, wrench schedules).  It contains none of the method's
arithmetic: no kinematics, dynamics, Philox parameter draws, predicates.  The
oracle (`oracle/`) and the product (`paper_2607_06337_b200/`) both receive the
arrays built here and share nothing else.

Recipes follow SURVEY.md section 8(d); DESIGN.md restates them.
"""
from .trees import (  # noqa: F401
    MASTER_SEED,
    WorldSpec,
    Params,
    binary_tree_config1,
    stochastic_world,
    ternary_lsystem_world,
    make_config,
    config_params,
)
from .loads import (  # noqa: F401
    config1_loads,
    config2_pulls,
    wrench_process,
    wrench_epoch_loads,
)
