"""FP64 CPU oracle of the f-x poststack depth-migration hot path -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from the CUDA package and shares no code with it.
"""
from .oracle import build, migrate, migrate_field, migrate_shot, migrate3d, table_index, num_threads  # noqa: F401
from .brute import brute_force_migrate  # noqa: F401
from .tf_oracle import section_to_fx  # noqa: F401
from . import design_oracle  # noqa: F401
