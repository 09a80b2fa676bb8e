"""CPU oracle for the Q-Render hot path -- TEST INFRASTRUCTURE ONLY (see qr_oracle.c header)."""
from . import qr_oracle  # noqa: F401
