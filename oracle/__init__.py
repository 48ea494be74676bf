"""CPU oracle for FPN RoIAlign.  TEST INFRASTRUCTURE: see raf_ref.cpp's header."""
