"""CPU oracle — TEST INFRASTRUCTURE ONLY.  See mcdc_oracle.h for the rules on who may import this."""
from .binding import Oracle, lib, COUNTER_NAMES  # noqa: F401
