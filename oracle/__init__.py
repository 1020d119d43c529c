"""CPU oracle of the EMC hot path -- test infrastructure only (see emc_oracle.py header)."""
from . import emc_oracle  # noqa: F401
