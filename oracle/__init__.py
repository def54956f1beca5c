"""CPU oracle of the seed x hit scan -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see comet_oracle.c)."""
from . import comet_oracle  # noqa: F401
