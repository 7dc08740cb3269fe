"""Oracle for the Nekbone CG hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see nko.h)."""
